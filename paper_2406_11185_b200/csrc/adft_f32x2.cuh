// adft_f32x2.cuh -- the single-precision class kernel of the mixed-precision dispatch,
// written for Blackwell's packed fp32 arithmetic: one lane evaluates TWO shell quartets (the same bra pair with two
// neighbouring ket pairs) whose recurrences run as one stream of FFMA2 / FMUL2 / FADD2 instructions on float2 operands
// (__ffma2_rn and friends, sm_100 and later).  The class kernels are bound by instruction issue, not by the FP32 pipe
// (ncu: 50-70% of the thread instructions of the low classes are not floating point at all, and a scalar fp32
// instantiation of the same code ran only 1.1-1.4x faster than fp64), so halving the number of arithmetic instructions
// per quartet is what single precision can buy here.
//
// The generated class code (csrc/generated/eri_*.cuh) is a template over the arithmetic type R; here R = F2.  What stays
// scalar per quartet: the geometry (the difference P - Q of the product centres in fp64), the Boys function (its table
// row depends on the quartet) and the reductions into J and K (fp64).
#pragma once
#include "adft_device.cuh"

namespace adft {

struct F2 {
    float2 v;
    __device__ __forceinline__ F2() {}
    __device__ __forceinline__ F2(int a) : v(make_float2((float)a, (float)a)) {}
    __device__ __forceinline__ F2(float a) : v(make_float2(a, a)) {}
    __device__ __forceinline__ F2(double a) : v(make_float2((float)a, (float)a)) {}
    __device__ __forceinline__ F2(float a, float b) : v(make_float2(a, b)) {}
};
__device__ __forceinline__ F2 operator*(F2 a, F2 b) { F2 r; r.v = __fmul2_rn(a.v, b.v); return r; }
__device__ __forceinline__ F2 operator+(F2 a, F2 b) { F2 r; r.v = __fadd2_rn(a.v, b.v); return r; }
__device__ __forceinline__ F2 operator-(F2 a) { return F2(-a.v.x, -a.v.y); }
__device__ __forceinline__ F2 operator-(F2 a, F2 b) { F2 r; r.v = __fadd2_rn(a.v, make_float2(-b.v.x, -b.v.y)); return r; }
__device__ __forceinline__ F2 &operator+=(F2 &a, F2 b) { a.v = __fadd2_rn(a.v, b.v); return a; }

// found by the unqualified fma(...) of the generated code (argument-dependent lookup) and by the accumulator classes
__device__ __forceinline__ F2 fma(F2 a, F2 b, F2 c) { F2 r; r.v = __ffma2_rn(a.v, b.v, c.v); return r; }
__device__ __forceinline__ F2 fma3(F2 a, F2 b, F2 c) { return fma(a, b, c); }

// primitive-pair record of this kernel: scalars in float, the product centre in double (PairTable::prim, primf)
struct PrimPairF {
    float zeta, inv2z, PAx, PAy, PAz, cc;
    double Px, Py, Pz;
};
__device__ __forceinline__ PrimPairF load_prim_f(const PairTable &t, int idx)
{
    const double *r = reinterpret_cast<const double *>(t.prim + (size_t)(idx >> 3) * 40 + (idx & 7));
    const float *f = t.primf + idx;
    const size_t n = t.primf_stride;
    PrimPairF p;
    p.zeta = __ldg(f);  p.inv2z = __ldg(f + n);
    p.PAx = __ldg(f + 2 * n);  p.PAy = __ldg(f + 3 * n);  p.PAz = __ldg(f + 4 * n);
    p.cc = __ldg(f + 5 * n);
    p.Px = __ldg(r + 16);  p.Py = __ldg(r + 17);  p.Pz = __ldg(r + 32);          // groups 1 and 2 of the fp64 record
    return p;
}

// One primitive quartet for each of the lane's two shell quartets: bra record b, ket records k0 and k1.
template <class V, class Acc>
__device__ __forceinline__ void prim_quartet2(const PrimPairF &b, const PrimPairF &k0, const PrimPairF &k1,
                                              const float *__restrict__ boys, Acc &acc, bool live0, bool live1)
{
    const float s0 = b.zeta + k0.zeta, s1 = b.zeta + k1.zeta;
    const float r0 = rsqrtf(s0), r1 = rsqrtf(s1);
    const F2 inv_s(r0 * r0, r1 * r1);
    PrimCtxT<F2> c;
    c.roz = F2(k0.zeta, k1.zeta) * inv_s;
    c.roe = F2(b.zeta) * inv_s;
    const F2 rho = F2(b.zeta) * c.roz;
    // P - Q in double: a difference of nearby coordinates
    const F2 PQx((float)(b.Px - k0.Px), (float)(b.Px - k1.Px)), PQy((float)(b.Py - k0.Py), (float)(b.Py - k1.Py)),
        PQz((float)(b.Pz - k0.Pz), (float)(b.Pz - k1.Pz));
    const F2 T = rho * fma(PQx, PQx, fma(PQy, PQy, PQz * PQz));
    const F2 mroz = -c.roz;
    c.WPx = mroz * PQx;  c.WPy = mroz * PQy;  c.WPz = mroz * PQz;
    c.WQx = c.roe * PQx;  c.WQy = c.roe * PQy;  c.WQz = c.roe * PQz;
    c.PAx = F2(b.PAx);  c.PAy = F2(b.PAy);  c.PAz = F2(b.PAz);
    c.QCx = F2(k0.PAx, k1.PAx);  c.QCy = F2(k0.PAy, k1.PAy);  c.QCz = F2(k0.PAz, k1.PAz);
    c.inv2z = F2(b.inv2z);  c.inv2e = F2(k0.inv2z, k1.inv2z);  c.inv2ze = F2(0.5f) * inv_s;
    // lanes or halves without a quartet go down the cheap asymptotic branch; their result has weight 0
    float Fa[V::MMAX + 1], Fb[V::MMAX + 1];
    boys_scaled_f<V::MMAX>(live0 ? T.v.x : 1.0e4f, b.cc * k0.cc * r0, boys, Fa);
    boys_scaled_f<V::MMAX>(live1 ? T.v.y : 1.0e4f, b.cc * k1.cc * r1, boys, Fb);
    F2 F[V::MMAX + 1];
#pragma unroll
    for (int m = 0; m <= V::MMAX; ++m) F[m] = F2(Fa[m], Fb[m]);
    V::vrr(c, F, acc);
}

template <class GP, int P, class Acc>
__device__ __forceinline__ void run_passes2(const PairTable &t, const Segment &sg, int i, int j0, int j1, bool live0, bool live1,
                                            const float *__restrict__ boys, Acc &acc)
{
    AccReg<GP::pass_nacc(P), F2> chunk;
    chunk.init(0, nullptr, 0, 0);
    for (int kb = 0; kb < sg.bra_K; ++kb) {
        const PrimPairF bp = load_prim_f(t, sg.bra_prim_base + kb * sg.bra_n + i);
        for (int kk = 0; kk < sg.ket_K; ++kk) {
            const PrimPairF kp0 = load_prim_f(t, sg.ket_prim_base + kk * sg.ket_n + j0);
            const PrimPairF kp1 = load_prim_f(t, sg.ket_prim_base + kk * sg.ket_n + j1);
            prim_quartet2<OnePass<GP, P>>(bp, kp0, kp1, boys, chunk, live0, live1);
        }
    }
    GP::template store_pass<P>(chunk, acc);
    if constexpr (P + 1 < GP::NPASS) run_passes2<GP, P + 1>(t, sg, i, j0, j1, live0, live1, boys, acc);
}

// (a5) digestion of the lane's two quartets (a b|c0 d0) and (a b|c1 d1): the six updates of DigestJK per quartet, the
// FMAs packed, D blocks pre-scaled by each quartet's own weight (0 for a half without a quartet), every reduction fp64.
template <class G>
struct DigestJK2 {
    static constexpr int NA = G::NA, NB = G::NB, NC = G::NC, ND = G::ND;
    F2 dab[NA * NB], dcd[NC * ND], dac[NA * NC], dad[NA * ND], dbc[NB * NC], dbd[NB * ND];
    F2 jab[NA * NB], jcd[NC * ND], kac[NA * NC], kad[NA * ND], kbc[NB * NC], kbd[NB * ND];

    __device__ __forceinline__ void load(const double *__restrict__ D, int N, int a0, int b0, int c0, int d0, int c1, int d1,
                                         double w0, double w1)
    {
#define ADFT_LD2(arr, n1, n2, r0_, q0_, r1_, q1_, f)                                                                       \
    _Pragma("unroll") for (int i = 0; i < n1; ++i) _Pragma("unroll") for (int j = 0; j < n2; ++j) {                        \
        arr[i * n2 + j] = F2((float)((f) * w0 * __ldg(D + (size_t)((r0_) + i) * N + (q0_) + j)),                           \
                             (float)((f) * w1 * __ldg(D + (size_t)((r1_) + i) * N + (q1_) + j)));                           \
    }
        ADFT_LD2(dab, NA, NB, a0, b0, a0, b0, 2.0)
        ADFT_LD2(dcd, NC, ND, c0, d0, c1, d1, 2.0)
        ADFT_LD2(dac, NA, NC, a0, c0, a0, c1, 1.0)
        ADFT_LD2(dad, NA, ND, a0, d0, a0, d1, 1.0)
        ADFT_LD2(dbc, NB, NC, b0, c0, b0, c1, 1.0)
        ADFT_LD2(dbd, NB, ND, b0, d0, b0, d1, 1.0)
#undef ADFT_LD2
#pragma unroll
        for (int i = 0; i < NA * NB; ++i) jab[i] = F2(0);
#pragma unroll
        for (int i = 0; i < NC * ND; ++i) jcd[i] = F2(0);
#pragma unroll
        for (int i = 0; i < NA * NC; ++i) kac[i] = F2(0);
#pragma unroll
        for (int i = 0; i < NA * ND; ++i) kad[i] = F2(0);
#pragma unroll
        for (int i = 0; i < NB * NC; ++i) kbc[i] = F2(0);
#pragma unroll
        for (int i = 0; i < NB * ND; ++i) kbd[i] = F2(0);
    }

    template <int ia, int ib, int ic, int id>
    __device__ __forceinline__ void put(F2 v)
    {
        jab[ia * NB + ib] = fma(dcd[ic * ND + id], v, jab[ia * NB + ib]);
        jcd[ic * ND + id] = fma(dab[ia * NB + ib], v, jcd[ic * ND + id]);
        kac[ia * NC + ic] = fma(dbd[ib * ND + id], v, kac[ia * NC + ic]);
        kad[ia * ND + id] = fma(dbc[ib * NC + ic], v, kad[ia * ND + id]);
        kbc[ib * NC + ic] = fma(dad[ia * ND + id], v, kbc[ib * NC + ic]);
        kbd[ib * ND + id] = fma(dac[ia * NC + ic], v, kbd[ib * ND + id]);
    }

    __device__ __forceinline__ void store(double *__restrict__ J, double *__restrict__ K, int N, int a0, int b0, int c0, int d0,
                                          int c1, int d1, bool v0, bool v1, int lane)
    {
#pragma unroll
        for (int i = 0; i < NA * NB; ++i) {                  // J_ab: both halves and the TILE_C lanes of the row share it
            double v = (double)jab[i].v.x + (double)jab[i].v.y;
#pragma unroll
            for (int o = TILE_C / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if ((lane & (TILE_C - 1)) == 0 && v != 0.0) atomicAdd(J + (size_t)(a0 + i / NB) * N + b0 + i % NB, v);
        }
        if (v0) {
#pragma unroll
            for (int i = 0; i < NC * ND; ++i) atomicAdd(J + (size_t)(c0 + i / ND) * N + d0 + i % ND, (double)jcd[i].v.x);
#pragma unroll
            for (int i = 0; i < NA * NC; ++i) atomicAdd(K + (size_t)(a0 + i / NC) * N + c0 + i % NC, (double)kac[i].v.x);
#pragma unroll
            for (int i = 0; i < NA * ND; ++i) atomicAdd(K + (size_t)(a0 + i / ND) * N + d0 + i % ND, (double)kad[i].v.x);
#pragma unroll
            for (int i = 0; i < NB * NC; ++i) atomicAdd(K + (size_t)(b0 + i / NC) * N + c0 + i % NC, (double)kbc[i].v.x);
#pragma unroll
            for (int i = 0; i < NB * ND; ++i) atomicAdd(K + (size_t)(b0 + i / ND) * N + d0 + i % ND, (double)kbd[i].v.x);
        }
        if (v1) {
#pragma unroll
            for (int i = 0; i < NC * ND; ++i) atomicAdd(J + (size_t)(c1 + i / ND) * N + d1 + i % ND, (double)jcd[i].v.y);
#pragma unroll
            for (int i = 0; i < NA * NC; ++i) atomicAdd(K + (size_t)(a0 + i / NC) * N + c1 + i % NC, (double)kac[i].v.y);
#pragma unroll
            for (int i = 0; i < NA * ND; ++i) atomicAdd(K + (size_t)(a0 + i / ND) * N + d1 + i % ND, (double)kad[i].v.y);
#pragma unroll
            for (int i = 0; i < NB * NC; ++i) atomicAdd(K + (size_t)(b0 + i / NC) * N + c1 + i % NC, (double)kbc[i].v.y);
#pragma unroll
            for (int i = 0; i < NB * ND; ++i) atomicAdd(K + (size_t)(b0 + i / ND) * N + d1 + i % ND, (double)kbd[i].v.y);
        }
    }
};

// A warp tile of this kernel is TILE_R bra pairs x 2*TILE_C ket pairs: lane (r, c) holds the ket pairs 2c and 2c+1 of the
// tile (Segment::tiles_per_row and col_tile_begin count tiles of that width; the host plan knows, adft_lib.cu).
constexpr int TILE_C2 = 2 * TILE_C;

template <class G, class GP, int ACCMODE, int WPB, int MINB>
__global__ void __launch_bounds__(WPB * 32, MINB) jk_kernel_f32x2(const JKParams p)
{
    extern __shared__ double s_acc_raw[];
    F2 *s_acc = reinterpret_cast<F2 *>(s_acc_raw);
    __shared__ unsigned long long s_cnt[3];
    __shared__ unsigned int s_done;
    if (threadIdx.x < 3) s_cnt[threadIdx.x] = 0ull;
    if (threadIdx.x == 3) s_done = 0u;
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const long long w = ((long long)blockIdx.x * WPB + (threadIdx.x >> 5)) * p.shard_count + p.shard_rank;
    if (w < p.total_warps) {
        const int lo = find_segment(p, w);
        const Segment sg = p.segs[lo];
        const long long r = w - sg.warp_begin;
        int i = sg.row_begin + (int)(r / sg.tiles_per_row) * TILE_R + lane / TILE_C;
        int j0 = ((int)(r % sg.tiles_per_row) + sg.col_tile_begin) * TILE_C2 + 2 * (lane & (TILE_C - 1));
        int j1 = j0 + 1;
        const int jend = sg.same ? (i + 1) : sg.ket_n;
        bool v0 = i < sg.rows && j0 < jend, v1 = i < sg.rows && j1 < jend;
        if (!v0) { i = 0; j0 = 0; }
        if (!v1) j1 = j0;
        const int gab = sg.bra_pair_base + i, gcd0 = sg.ket_pair_base + j0, gcd1 = sg.ket_pair_base + j1;
        const double Qab = __ldg(p.t.Q + gab);
        // the band test of the mixed-precision dispatch (R-24), per quartet: tau <= S < tau_hi
        const double S0 = (Qab * __ldg(p.t.Q + gcd0)) * screen_density(p, gab, gcd0);
        const double S1 = (Qab * __ldg(p.t.Q + gcd1)) * screen_density(p, gab, gcd1);
        v0 = v0 && S0 >= p.tau && S0 < p.tau_hi;
        v1 = v1 && S1 >= p.tau && S1 < p.tau_hi;
        const unsigned b0m = __ballot_sync(0xffffffffu, v0), b1m = __ballot_sync(0xffffffffu, v1);
        if ((b0m | b1m) != 0u) {
            const unsigned kab = (unsigned)__ldg(p.t.knom + gab);
            const unsigned knom = __reduce_add_sync(0xffffffffu, (v0 ? kab * (unsigned)__ldg(p.t.knom + gcd0) : 0u)
                                                                     + (v1 ? kab * (unsigned)__ldg(p.t.knom + gcd1) : 0u));
            if (lane == 0) {
                const unsigned long long n = (unsigned long long)(__popc(b0m) + __popc(b1m));
                atomicAdd(&s_cnt[0], n);
                atomicAdd(&s_cnt[1], n * (unsigned long long)(sg.bra_K * sg.ket_K));
                atomicAdd(&s_cnt[2], (unsigned long long)knom);
            }
            typename AccSel<ACCMODE, G::NACC, F2>::type acc;
            if constexpr (GP::NPASS == 1) {
                acc.init(p.zero, s_acc, threadIdx.x, WPB * 32);
                for (int kb = 0; kb < sg.bra_K; ++kb) {
                    const PrimPairF bp = load_prim_f(p.t, sg.bra_prim_base + kb * sg.bra_n + i);
                    for (int kk = 0; kk < sg.ket_K; ++kk) {
                        const PrimPairF kp0 = load_prim_f(p.t, sg.ket_prim_base + kk * sg.ket_n + j0);
                        const PrimPairF kp1 = load_prim_f(p.t, sg.ket_prim_base + kk * sg.ket_n + j1);
                        prim_quartet2<SinglePass<G>>(bp, kp0, kp1, p.boys_f, acc, v0, v1);
                    }
                }
            } else {
                acc.bind(p.zero, s_acc, threadIdx.x, WPB * 32);
                run_passes2<GP, 0>(p.t, sg, i, j0, j1, v0, v1, p.boys_f, acc);
            }
            const int sa = __ldg(p.t.sha + gab), sb = __ldg(p.t.shb + gab);
            double w0 = v0 ? 1.0 : 0.0, w1 = v1 ? 1.0 : 0.0;
            if (sa == sb) { w0 *= 0.5; w1 *= 0.5; }
            if (__ldg(p.t.sha + gcd0) == __ldg(p.t.shb + gcd0)) w0 *= 0.5;
            if (__ldg(p.t.sha + gcd1) == __ldg(p.t.shb + gcd1)) w1 *= 0.5;
            if (gab == gcd0) w0 *= 0.5;
            if (gab == gcd1) w1 *= 0.5;
            const int a0 = __ldg(p.t.bfa + gab), b0 = __ldg(p.t.bfb + gab);
            const int c0 = __ldg(p.t.bfa + gcd0), d0 = __ldg(p.t.bfb + gcd0);
            const int c1 = __ldg(p.t.bfa + gcd1), d1 = __ldg(p.t.bfb + gcd1);
            DigestJK2<G> dg;
            dg.load(p.D, p.N, a0, b0, c0, d0, c1, d1, w0, w1);
            G::hrr(acc, F2((float)__ldg(p.t.ABx + gab)), F2((float)__ldg(p.t.ABy + gab)), F2((float)__ldg(p.t.ABz + gab)),
                   F2((float)__ldg(p.t.ABx + gcd0), (float)__ldg(p.t.ABx + gcd1)),
                   F2((float)__ldg(p.t.ABy + gcd0), (float)__ldg(p.t.ABy + gcd1)),
                   F2((float)__ldg(p.t.ABz + gcd0), (float)__ldg(p.t.ABz + gcd1)), dg);
            dg.store(p.J, p.K, p.N, a0, b0, c0, d0, c1, d1, v0, v1, lane);
        }
    }
    if (lane == 0) {
        __threadfence_block();
        if (atomicAdd(&s_done, 1u) == WPB - 1) {
            __threadfence_block();
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const unsigned long long v = atomicAdd(&s_cnt[c], 0ull);
                if (v) atomicAdd(p.counters + c, v);
            }
        }
    }
}

template <class G, class GP, int ACCMODE, int WPB, int MINB>
inline void launch_jk_f32x2(const JKParams &p, cudaStream_t st)
{
    const long long mine = (p.total_warps - p.shard_rank + p.shard_count - 1) / p.shard_count;
    if (mine <= 0) return;
    const unsigned nb = (unsigned)((mine + WPB - 1) / WPB);
    const size_t smem = ACCMODE == ACC_SMEM ? (size_t)G::NACC * WPB * 32 * sizeof(F2) : 0;
    auto kern = jk_kernel_f32x2<G, GP, ACCMODE, WPB, MINB>;
    if (smem > 48 * 1024) cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    kern<<<nb, WPB * 32, smem, st>>>(p);
}


// all four kernels of a class behind one call (tuning builds instantiate them in one translation unit)
template <class G, class GP, int ACCMODE, int WPB, int MINB>
inline void launch_jk_class(const JKParams &p, cudaStream_t st, bool want_j, bool want_k, bool fp32)
{
    if (fp32) launch_jk_f32x2<G, GP, ACCMODE, WPB, MINB>(p, st);
    else if (want_j && want_k) launch_jk_variant<G, GP, true, true, ACCMODE, WPB, MINB>(p, st);
    else if (want_j) launch_jk_variant<G, GP, true, false, ACCMODE, WPB, MINB>(p, st);
    else launch_jk_variant<G, GP, false, true, ACCMODE, WPB, MINB>(p, st);
}

}  // namespace adft
