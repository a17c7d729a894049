// adft_interp.cuh -- table-driven class kernels: the same Obara-Saika/HGP recurrence DAGs the generator emits as
// straight-line code (csrc/gen/gen_eri.py), serialised as int32 instruction lists and executed by a per-lane
// interpreter.  Used for the quartet classes whose [e0|f0] block is too large for registers / straight-line code
// (the classes with f shells, up to (ff|ff): 5476 contracted accumulators, 22208 recurrence steps per primitive
// quartet).  One lane = one shell quartet, exactly as in jk_kernel; the per-lane working set (recurrence slots,
// contracted accumulators, HRR slots, D/J/K blocks) lives in a global scratch buffer laid out slot-major
// (element q of thread t at scratch[q*stride + t]) so that a warp's access to one slot is one coalesced 256-byte line.
// The kernel is persistent (a few CTAs per SM) and warps fetch tiles from an atomic counter, the device-side
// analogue of the paper's global task counter.
#pragma once
#include "adft_device.cuh"

namespace adft {

// instruction kinds of the VRR program (gen_eri.py: K_B .. K_ACC)
enum { IK_B = 0, IK_TBRA = 1, IK_TKET = 2, IK_A = 3, IK_K = 4, IK_ACC = 5 };

struct InterpProg {
    const int4 *vrr;          // [n_vrr][2]: (op|dir<<4, dst, s0, s1), (s2, s3, n2, nx)
    const int4 *hrr;          // [n_hrr]: (which|dir<<2, dst, k0, k1); which 2 = output (dst = packed components, k0 = src)
    int32_t n_vrr, n_hrr, n_vslots, n_hslots, nacc, mmax;
    int32_t la, lb, lc, ld;
};

struct InterpParams {
    JKParams jk;
    InterpProg prog;
    double *scratch;                  // [nslots][stride]
    long long stride;                 // threads of the persistent grid
    unsigned long long *tile_counter; // zeroed before the launch
    const double *boys_plain;         // F_m(T_k) table [BOYS_NT][BOYS_NM] (boys_scaled_rt)
};

__host__ __device__ inline int interp_ncart(int l) { return (l + 1) * (l + 2) / 2; }

// scratch slots needed per thread by the J/K kernel of a class
inline int interp_jk_slots(int n_vslots, int n_hslots, int nacc, int la, int lb, int lc, int ld)
{
    const int na = interp_ncart(la), nb = interp_ncart(lb), nc = interp_ncart(lc), nd = interp_ncart(ld);
    const int blocks = 2 * (na * nb + nc * nd + na * nc + na * nd + nb * nc + nb * nd);
    const int phase2 = n_hslots + blocks;
    return nacc + (n_vslots > phase2 ? n_vslots : phase2);
}

// Boys function with a run-time order (same arithmetic as boys_scaled<MMAX>)
__device__ __forceinline__ void boys_scaled_rt(int mmax, double T, double pref, const double *__restrict__ tab, double *F)
{
    if (T < BOYS_TMAX) {
        const int k = __double2int_rn(T * 8.0);
        const double d = fma((double)k, 0.125, -T);
        const double *row = tab + k * BOYS_NM + mmax;
        double s = __ldg(row + 9);
        s = fma(s, d * (1.0 / 9.0), __ldg(row + 8));
        s = fma(s, d * (1.0 / 8.0), __ldg(row + 7));
        s = fma(s, d * (1.0 / 7.0), __ldg(row + 6));
        s = fma(s, d * (1.0 / 6.0), __ldg(row + 5));
        s = fma(s, d * (1.0 / 5.0), __ldg(row + 4));
        s = fma(s, d * (1.0 / 4.0), __ldg(row + 3));
        s = fma(s, d * (1.0 / 3.0), __ldg(row + 2));
        s = fma(s, d * (1.0 / 2.0), __ldg(row + 1));
        s = fma(s, d, __ldg(row));
        F[mmax] = s * pref;
        if (mmax > 0) {
            const double e = exp(-T) * pref;
            const double T2 = T + T;
            for (int m = mmax; m >= 1; --m) F[m - 1] = fma(T2, F[m], e) * (1.0 / (double)(2 * m - 1));
        }
    } else {
        const double r = rsqrt(T);
        F[0] = 0.88622692545275801365 * r * pref;
        const double h = 0.5 * r * r;
        for (int m = 1; m <= mmax; ++m) F[m] = F[m - 1] * ((double)(2 * m - 1) * h);
    }
}

__device__ __forceinline__ double sel3(int dir, double x, double y, double z) { return dir == 0 ? x : (dir == 1 ? y : z); }

// One primitive quartet through the VRR program; v slots at S[0..), accumulators at A[0..) (both strided).
__device__ __forceinline__ void interp_prim_quartet(const InterpProg &pg, const PrimPair &b, const PrimPair &k,
                                                    const double *__restrict__ boys, double *__restrict__ S,
                                                    double *__restrict__ A, long long stride)
{
    const double s = b.zeta + k.zeta;
    const double r = rsqrt(s);
    const double inv_s = r * r;
    const double roz = k.zeta * inv_s, roe = b.zeta * inv_s;
    const double rho = b.zeta * roz;
    const double PQx = b.Px - k.Px, PQy = b.Py - k.Py, PQz = b.Pz - k.Pz;
    const double T = rho * fma(PQx, PQx, fma(PQy, PQy, PQz * PQz));
    const double WPx = -roz * PQx, WPy = -roz * PQy, WPz = -roz * PQz;
    const double WQx = roe * PQx, WQy = roe * PQy, WQz = roe * PQz;
    const double inv2z = b.inv2z, inv2e = k.inv2z, inv2ze = 0.5 * inv_s;
    double F[16];
    boys_scaled_rt(pg.mmax, T, b.cc * k.cc * r, boys, F);
    const int4 *pv = pg.vrr;
    int4 a = __ldg(pv), c = __ldg(pv + 1);
    for (int i = 0; i < pg.n_vrr; ++i) {
        const int4 an = __ldg(pv + 2 * i + 2), cn = __ldg(pv + 2 * i + 3);     // the list is padded by one instruction
        const int kind = a.x & 15, dir = (a.x >> 4) & 3;
        if (kind == IK_A) {
            double e = fma(sel3(dir, b.PAx, b.PAy, b.PAz), S[a.z * stride], sel3(dir, WPx, WPy, WPz) * S[a.w * stride]);
            if (c.x >= 0) e = fma((double)c.z * inv2z, S[c.x * stride], e);
            S[a.y * stride] = e;
        } else if (kind == IK_K) {
            double e = fma(sel3(dir, k.PAx, k.PAy, k.PAz), S[a.z * stride], sel3(dir, WQx, WQy, WQz) * S[a.w * stride]);
            if (c.x >= 0) e = fma((double)c.z * inv2e, S[c.x * stride], e);
            if (c.y >= 0) e = fma((double)c.w * inv2ze, S[c.y * stride], e);
            S[a.y * stride] = e;
        } else if (kind == IK_ACC) {
            A[c.z * stride] += S[a.z * stride];
        } else if (kind == IK_TBRA) {
            S[a.y * stride] = fma(-roz, S[a.w * stride], S[a.z * stride]);
        } else if (kind == IK_TKET) {
            S[a.y * stride] = fma(-roe, S[a.w * stride], S[a.z * stride]);
        } else {
            S[a.y * stride] = F[a.z];
        }
        a = an; c = cn;
    }
}

__global__ void __launch_bounds__(128) jk_interp_kernel(const InterpParams q)
{
    const JKParams &p = q.jk;
    const InterpProg &pg = q.prog;
    const int lane = threadIdx.x & 31;
    const long long gtid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long st = q.stride;
    const int na = interp_ncart(pg.la), nb = interp_ncart(pg.lb), nc = interp_ncart(pg.lc), nd = interp_ncart(pg.ld);
    double *A = q.scratch + gtid;                          // contracted accumulators [nacc]
    double *S = A + (long long)pg.nacc * st;               // VRR slots, later HRR slots + blocks
    double *H = S;
    double *dab = H + (long long)pg.n_hslots * st, *dcd = dab + (long long)na * nb * st, *dac = dcd + (long long)nc * nd * st,
           *dad = dac + (long long)na * nc * st, *dbc = dad + (long long)na * nd * st, *dbd = dbc + (long long)nb * nc * st;
    double *jab = dbd + (long long)nb * nd * st, *jcd = jab + (long long)na * nb * st, *kac = jcd + (long long)nc * nd * st,
           *kad = kac + (long long)na * nc * st, *kbc = kad + (long long)na * nd * st, *kbd = kbc + (long long)nb * nc * st;
    unsigned long long cnt_q = 0ull, cnt_p = 0ull, cnt_n = 0ull;
    for (;;) {
        long long w = 0;
        if (lane == 0) w = (long long)atomicAdd(q.tile_counter, 1ull);
        w = __shfl_sync(0xffffffffu, w, 0);
        if (w >= p.total_warps) break;
        int lo = 0, hi = p.nsegs - 1;
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (__ldg(&p.segs[mid].warp_begin) <= w) lo = mid; else hi = mid - 1;
        }
        const Segment sg = p.segs[lo];
        const long long r = w - sg.warp_begin;
        int i = (int)(r / sg.tiles_per_row) * TILE_R + lane / TILE_C;
        int j = (int)(r % sg.tiles_per_row) * TILE_C + (lane & (TILE_C - 1));
        bool valid = i < sg.rows && j < (sg.same ? (i + 1) : sg.ket_n);
        if (!valid) { i = 0; j = 0; }
        const int gab = sg.bra_pair_base + i;
        const double Qab = __ldg(p.t.Q + gab);
        const int gcd = sg.ket_pair_base + j;
        valid = valid && ((Qab * __ldg(p.t.Q + gcd)) * p.dmax >= p.tau);      // the screen (DESIGN R-7)
        const unsigned ballot = __ballot_sync(0xffffffffu, valid);
        if (ballot == 0u) continue;
        const unsigned knom = __reduce_add_sync(0xffffffffu, valid ? (unsigned)(__ldg(p.t.knom + gab) * __ldg(p.t.knom + gcd)) : 0u);
        if (lane == 0) {
            const unsigned long long n = (unsigned long long)__popc(ballot);
            cnt_q += n;
            cnt_p += n * (unsigned long long)(sg.bra_K * sg.ket_K);
            cnt_n += (unsigned long long)knom;
        }
        for (int x = 0; x < pg.nacc; ++x) A[x * st] = 0.0;
        for (int kb = 0; kb < sg.bra_K; ++kb) {
            const PrimPair bp = load_prim(p.t, sg.bra_prim_base + kb * sg.bra_n + i);
            for (int kk = 0; kk < sg.ket_K; ++kk) {
                const PrimPair kp = load_prim(p.t, sg.ket_prim_base + kk * sg.ket_n + j);
                interp_prim_quartet(pg, bp, kp, q.boys_plain, S, A, st);
            }
        }
        // D blocks (weight folded in) and zeroed J/K blocks
        const int sa = __ldg(p.t.sha + gab), sb = __ldg(p.t.shb + gab);
        const int sc = __ldg(p.t.sha + gcd), sd = __ldg(p.t.shb + gcd);
        double wgt = valid ? 1.0 : 0.0;
        if (sa == sb) wgt *= 0.5;
        if (sc == sd) wgt *= 0.5;
        if (gab == gcd) wgt *= 0.5;
        const int a0 = __ldg(p.t.bfa + gab), b0 = __ldg(p.t.bfb + gab);
        const int c0 = __ldg(p.t.bfa + gcd), d0 = __ldg(p.t.bfb + gcd);
        const double *D = p.D;
        const int N = p.N;
        const double w2 = wgt + wgt;
        for (int x = 0; x < na; ++x) for (int y = 0; y < nb; ++y) { dab[(x * nb + y) * st] = w2 * __ldg(D + (size_t)(a0 + x) * N + b0 + y); jab[(x * nb + y) * st] = 0.0; }
        for (int x = 0; x < nc; ++x) for (int y = 0; y < nd; ++y) { dcd[(x * nd + y) * st] = w2 * __ldg(D + (size_t)(c0 + x) * N + d0 + y); jcd[(x * nd + y) * st] = 0.0; }
        for (int x = 0; x < na; ++x) for (int y = 0; y < nc; ++y) { dac[(x * nc + y) * st] = wgt * __ldg(D + (size_t)(a0 + x) * N + c0 + y); kac[(x * nc + y) * st] = 0.0; }
        for (int x = 0; x < na; ++x) for (int y = 0; y < nd; ++y) { dad[(x * nd + y) * st] = wgt * __ldg(D + (size_t)(a0 + x) * N + d0 + y); kad[(x * nd + y) * st] = 0.0; }
        for (int x = 0; x < nb; ++x) for (int y = 0; y < nc; ++y) { dbc[(x * nc + y) * st] = wgt * __ldg(D + (size_t)(b0 + x) * N + c0 + y); kbc[(x * nc + y) * st] = 0.0; }
        for (int x = 0; x < nb; ++x) for (int y = 0; y < nd; ++y) { dbd[(x * nd + y) * st] = wgt * __ldg(D + (size_t)(b0 + x) * N + d0 + y); kbd[(x * nd + y) * st] = 0.0; }
        // HRR program with interleaved outputs; every output is digested at once (a5)
        const double ABx = __ldg(p.t.ABx + gab), ABy = __ldg(p.t.ABy + gab), ABz = __ldg(p.t.ABz + gab);
        const double CDx = __ldg(p.t.ABx + gcd), CDy = __ldg(p.t.ABy + gcd), CDz = __ldg(p.t.ABz + gcd);
        const int4 *ph = pg.hrr;
        int4 a = __ldg(ph);
        for (int x = 0; x < pg.n_hrr; ++x) {
            const int4 an = __ldg(ph + x + 1);                                   // padded by one instruction
            const int which = a.x & 3, dir = (a.x >> 2) & 3;
            const double v0 = a.z < 0 ? A[(long long)(-a.z - 1) * st] : H[a.z * st];
            if (which == 2) {
                const int ia = a.y & 255, ib = (a.y >> 8) & 255, ic = (a.y >> 16) & 255, id = (a.y >> 24) & 255;
                jab[(ia * nb + ib) * st] = fma(dcd[(ic * nd + id) * st], v0, jab[(ia * nb + ib) * st]);
                jcd[(ic * nd + id) * st] = fma(dab[(ia * nb + ib) * st], v0, jcd[(ic * nd + id) * st]);
                kac[(ia * nc + ic) * st] = fma(dbd[(ib * nd + id) * st], v0, kac[(ia * nc + ic) * st]);
                kad[(ia * nd + id) * st] = fma(dbc[(ib * nc + ic) * st], v0, kad[(ia * nd + id) * st]);
                kbc[(ib * nc + ic) * st] = fma(dad[(ia * nd + id) * st], v0, kbc[(ib * nc + ic) * st]);
                kbd[(ib * nd + id) * st] = fma(dac[(ia * nc + ic) * st], v0, kbd[(ib * nd + id) * st]);
            } else {
                const double v1 = a.w < 0 ? A[(long long)(-a.w - 1) * st] : H[a.w * st];
                const double g = which == 0 ? sel3(dir, ABx, ABy, ABz) : sel3(dir, CDx, CDy, CDz);
                H[a.y * st] = fma(g, v1, v0);
            }
            a = an;
        }
        // stores: J_ab is common to the warp (shuffle-reduce, one atomic per element); the rest is lane-private
        double *J = p.J, *K = p.K;
        for (int x = 0; x < na * nb; ++x) {
            double v = jab[x * st];
            for (int o = TILE_C / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if ((lane & (TILE_C - 1)) == 0 && v != 0.0) atomicAdd(J + (size_t)(a0 + x / nb) * N + b0 + x % nb, v);
        }
        if (valid) {
            for (int x = 0; x < nc * nd; ++x) atomicAdd(J + (size_t)(c0 + x / nd) * N + d0 + x % nd, jcd[x * st]);
            for (int x = 0; x < na * nc; ++x) atomicAdd(K + (size_t)(a0 + x / nc) * N + c0 + x % nc, kac[x * st]);
            for (int x = 0; x < na * nd; ++x) atomicAdd(K + (size_t)(a0 + x / nd) * N + d0 + x % nd, kad[x * st]);
            for (int x = 0; x < nb * nc; ++x) atomicAdd(K + (size_t)(b0 + x / nc) * N + c0 + x % nc, kbc[x * st]);
            for (int x = 0; x < nb * nd; ++x) atomicAdd(K + (size_t)(b0 + x / nd) * N + d0 + x % nd, kbd[x * st]);
        }
    }
    if (lane == 0 && cnt_q) {
        atomicAdd(p.counters, cnt_q);
        atomicAdd(p.counters + 1, cnt_p);
        atomicAdd(p.counters + 2, cnt_n);
    }
}

// (a2) Schwarz bounds through the diagonal HRR program of class (ab|ab); one thread per pair of a batch of at most
// `stride` pairs.  prog.hrr points at the diag program here.
__global__ void __launch_bounds__(128) schwarz_interp_kernel(PairTable t, InterpProg pg, int pair_base, int prim_base, int n,
                                                             int K, int first, int count, const double *__restrict__ boys,
                                                             double *__restrict__ Qout, double *scratch, long long st)
{
    const int tid = blockIdx.x * blockDim.x + threadIdx.x;
    if (tid >= count) return;
    const int j = first + tid;
    double *A = scratch + tid;
    double *S = A + (long long)pg.nacc * st;
    double *H = S;
    for (int x = 0; x < pg.nacc; ++x) A[x * st] = 0.0;
    for (int kb = 0; kb < K; ++kb) {
        const PrimPair bp = load_prim(t, prim_base + kb * n + j);
        for (int kk = 0; kk < K; ++kk) {
            const PrimPair kp = load_prim(t, prim_base + kk * n + j);
            interp_prim_quartet(pg, bp, kp, boys, S, A, st);
        }
    }
    const int g = pair_base + j;
    const double ABx = t.ABx[g], ABy = t.ABy[g], ABz = t.ABz[g];
    double mx = 0.0;
    const int4 *ph = pg.hrr;
    int4 a = __ldg(ph);
    for (int x = 0; x < pg.n_hrr; ++x) {
        const int4 an = __ldg(ph + x + 1);
        const int which = a.x & 3, dir = (a.x >> 2) & 3;
        const double v0 = a.z < 0 ? A[(long long)(-a.z - 1) * st] : H[a.z * st];
        if (which == 2) {
            mx = fmax(mx, fabs(v0));
        } else {
            const double v1 = a.w < 0 ? A[(long long)(-a.w - 1) * st] : H[a.w * st];
            H[a.y * st] = fma(sel3(dir, ABx, ABy, ABz), v1, v0);       // bra and ket of (ab|ab) share A-B
        }
        a = an;
    }
    Qout[g] = sqrt(mx);
}

}  // namespace adft
