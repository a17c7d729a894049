// adft_rys.cuh -- block-cooperative Rys-quadrature class kernels for the high-L quartet classes (f shells).
//
// Row (a4)/(a5) of SURVEY.md section 8 for the classes whose [e0|f0] block is too large for one lane
// ((fp|fp) ... (ff|ff): 625 ... 5476 contracted intermediates).  PAPER.md:72 names Rys quadrature beside HGP as the
// two methods its ERI code implements; here (Dupuis, Rys, King 1976; Rys, Dupuis, King 1983)
//     (ab|cd) = sum over primitive quartets, sum over roots r = 1..NR, NR = (la+lb+lc+ld)/2 + 1 of
//               Ix(ax,bx,cx,dx; r) * Iy(ay,by,cy,dy; r) * Iz(az,bz,cz,dz; r)
// with 2-D integrals from the recurrences (u = t_r^2, the Rys root; s = zeta+eta; rho = zeta eta / s)
//     B00 = u/(2s)   B10 = (1 - (rho/zeta) u)/(2 zeta)   B01 = (1 - (rho/eta) u)/(2 eta)
//     C00 = (P-A) - (rho/zeta) u (P-Q)      C00' = (Q-C) + (rho/eta) u (P-Q)
//     g[n+1][0] = C00 g[n][0] + n B10 g[n-1][0]
//     g[n][m+1] = C00' g[n][m] + m B01 g[n][m-1] + n B00 g[n-1][m]
// (the Obara-Saika vertical recurrence of SURVEY.md 8(c) with [..]^(m) = sum_r w_r u_r^m Ix Iy Iz), followed by the
// horizontal transfer in 2-D:  G(i,j+1;k,l) = G(i+1,j;k,l) + (A-B) G(i,j;k,l), likewise for (k,l) with (C-D).
//
// Mapping to the machine: ONE thread block works on one shell quartet at a time.
//   phase 1: thread (item, axis), item = (primitive quartet, root): roots/weights from the Chebyshev tables
//            (csrc/gen/gen_rys.py), the 2-D recurrences, result G[axis][i][j][k][l] to shared memory;
//   phase 2: thread (ab component pair, chunk of cd component pairs) keeps its contracted integrals in REGISTERS and
//            accumulates  acc += Gx*Gy*Gz  over the items of the batch: 3 shared-memory loads per (k,l) slot feed
//            all integrals of the chunk (1 DMUL + 1 DFMA each, operands in registers);
//   digestion (a5): the thread owns final integrals (ab|cd): J_ab by a private sum, J_cd by a warp shuffle reduction
//            (the lanes of a warp share the cd chunk), the four K blocks by private partial sums; one fp64 reduction
//            to global per touched element.
// Tiles (bra pair x 32 ket pairs, the same Segment table as jk_kernel) are fetched from an atomic counter.
#pragma once
#include <utility>
#include "adft_device.cuh"

namespace adft {

constexpr int RYS_NMAX = 9;   // roots of the largest class: (gg|gg), L = 16, L/2 + 1 = 9
struct RysTable {
    const double *tab;        // device copy of generated/rys_tables.bin (gen_rys.py layout)
    int32_t nint, ncoef;      // intervals on [0, tmax), Chebyshev coefficients per function
    double tmax, inv_h;
    int32_t off_cheb[RYS_NMAX + 1];      // [N]: start of the Chebyshev block of the N-point rule (doubles)
    int32_t off_asym[RYS_NMAX + 1];      // [N]: start of x_i^2 (N values) then h_i (N values)
};

// Root r (0-based, ascending) of the NR-point rule: u = t^2 and weight w.
template <int NR>
__device__ __forceinline__ void rys_root(const RysTable &rt, double T, int r, double &u, double &w)
{
    if (T < rt.tmax) {
        int k = (int)(T * rt.inv_h);
        k = k < rt.nint - 1 ? k : rt.nint - 1;
        const double x = 2.0 * fma(T, rt.inv_h, -(double)k) - 1.0;
        const double x2 = x + x;
        const double *cu = rt.tab + rt.off_cheb[NR] + ((size_t)k * 2 * NR + r) * rt.ncoef;
        const double *cw = cu + (size_t)NR * rt.ncoef;
        double b1 = 0.0, b2 = 0.0, d1 = 0.0, d2 = 0.0;
        for (int j = rt.ncoef - 1; j >= 1; --j) {           // Clenshaw
            const double t1 = fma(x2, b1, __ldg(cu + j) - b2);  b2 = b1;  b1 = t1;
            const double t2 = fma(x2, d1, __ldg(cw + j) - d2);  d2 = d1;  d1 = t2;
        }
        u = fma(x, b1, __ldg(cu) - b2);
        w = fma(x, d1, __ldg(cw) - d2);
    } else {
        const double ri = rsqrt_normal(T);
        u = __ldg(rt.tab + rt.off_asym[NR] + r) * ri * ri;
        w = __ldg(rt.tab + rt.off_asym[NR] + NR + r) * ri;
    }
}

__host__ __device__ constexpr int rys_ncart(int l) { return (l + 1) * (l + 2) / 2; }
// exponent of axis `ax` of Cartesian component `idx` of a shell with angular momentum l (order: lx descending, then ly)
__host__ __device__ constexpr int rys_cart(int l, int idx, int ax)
{
    int n = 0;
    for (int lx = l; lx >= 0; --lx)
        for (int ly = l - lx; ly >= 0; --ly) {
            if (n == idx) return ax == 0 ? lx : (ax == 1 ? ly : l - lx - ly);
            ++n;
        }
    return 0;
}
// run-time version: component idx of a shell with angular momentum L sits in row ii = L - lx of the triangle
// (rows of 1, 2, 3, ... components), ly = ii - (idx - ii(ii+1)/2)
template <int L>
__device__ __forceinline__ int rys_cart_rt(int idx, int ax)
{
    int ii = 0;
#pragma unroll
    for (int r = 1; r <= L; ++r) ii += (idx >= r * (r + 1) / 2) ? 1 : 0;
    const int lx = L - ii, ly = ii - (idx - ii * (ii + 1) / 2);
    return ax == 0 ? lx : (ax == 1 ? ly : L - lx - ly);
}

// Compile-time description of one class and its thread mapping.
// NCH thread groups work on NCH chunks of cd component pairs at a time; NPASS > 1 repeats both phases for further chunks
// (the g classes: (gg|gg) has 225 x 225 integrals per quartet, more than one block can hold in registers at once).
template <int LA_, int LB_, int LC_, int LD_, int NCH_, int NPASS_ = 1>
struct RysCfg {
    static constexpr int LA = LA_, LB = LB_, LC = LC_, LD = LD_, NCH = NCH_, NPASS = NPASS_;
    static constexpr int NCHT = NCH * NPASS;                       // cd chunks in total
    static constexpr int NR = (LA + LB + LC + LD) / 2 + 1;
    static constexpr int NA = rys_ncart(LA), NB = rys_ncart(LB), NC = rys_ncart(LC), ND = rys_ncart(LD);
    static constexpr int NAB = NA * NB, NCD = NC * ND;
    static constexpr int NABP = (NAB + 31) / 32 * 32;
    static constexpr int NT = NCH * NABP;                          // threads per block
    static constexpr int CH = (NCD + NCHT - 1) / NCHT;             // cd component pairs per thread and pass
    static constexpr int NKL = (LC + 1) * (LD + 1);
    static constexpr int PADCD = NKL | 1;                          // odd stride: the (i,j) slots fall in distinct banks
    // doubles per (item, axis), odd: in phase 1 the 16 lanes of a 64-bit shared-memory wavefront write the same slot of
    // 16 consecutive (item, axis) units, AXSZ doubles apart; an even AXSZ folds them onto a few banks (ncu, (fd|dp) with
    // AXSZ = 84: 31% of all shared-memory wavefronts were bank-conflict replays, L1/TEX at 91% of peak)
    static constexpr int AXSZ = ((LA + 1) * (LB + 1) * PADCD) | 1;
    static constexpr int ITEMSZ = 3 * AXSZ;                        // doubles per (primitive quartet, root)
    // shared memory per block: one big block per SM for the largest classes, several small blocks per SM otherwise
    static constexpr int SMEM_BUDGET = ITEMSZ * 8 > 4096 ? 196 * 1024 : (NT <= 64 ? 32 * 1024 : 64 * 1024);
    static constexpr int BATCH_S = SMEM_BUDGET / (ITEMSZ * 8);
    static constexpr int BATCH = BATCH_S < 64 ? BATCH_S : 64;      // phase 1 strides over 3*BATCH units with NT threads
    static constexpr size_t SMEM_BYTES = (size_t)BATCH * ITEMSZ * 8;
    static constexpr int MINB = NT <= 64 ? 6 : (NT <= 128 ? 3 : 1);   // resident blocks per SM asked of the register allocator
};

// phase 1: the 2-D integrals of one (primitive quartet, root, axis), all (i<=la, j<=lb, k<=lc, l<=ld), to `out`
// (layout out[(i*(LB+1)+j)*PADCD + k*(LD+1)+l]).  The z axis carries prefactor * weight.
// Recurrence centre (R-22): the vertical recurrence is built on whichever shell of the pair is nearer to
// this primitive pair's product centre (B instead of A iff |P-B| < |P-A|, D instead of C iff |Q-D| < |Q-C|) and the
// horizontal transfer runs towards the other shell, so the transferred factor (x - far centre) = (x - near centre) +
// (near - far) never has to cancel a large recurrence value.  The choice costs nothing here because the transfer is
// done per primitive in 2-D.
template <class C>
__device__ __forceinline__ void rys_phase1(const RysTable &rt, const PrimPair &b, const PrimPair &k, int r, int ax,
                                           const double (&ABv)[3], const double (&CDv)[3], double *__restrict__ out)
{
    constexpr int NBR = C::LA + C::LB, NKT = C::LC + C::LD;
    const double s = b.zeta + k.zeta;
    const double rs = rsqrt_normal(s);
    const double inv_s = rs * rs;
    const double roz = k.zeta * inv_s, roe = b.zeta * inv_s;      // rho/zeta, rho/eta
    const double rho = b.zeta * roz;
    const double PQx = b.Px - k.Px, PQy = b.Py - k.Py, PQz = b.Pz - k.Pz;
    const double T = rho * fma(PQx, PQx, fma(PQy, PQy, PQz * PQz));
    double u, w;
    rys_root<C::NR>(rt, T, r, u, w);
    const double pq = ax == 0 ? PQx : (ax == 1 ? PQy : PQz);
    const double PBx = b.PAx + ABv[0], PBy = b.PAy + ABv[1], PBz = b.PAz + ABv[2];       // P - B
    const double QDx = k.PAx + CDv[0], QDy = k.PAy + CDv[1], QDz = k.PAz + CDv[2];       // Q - D
    const bool onB = fma(PBx, PBx, fma(PBy, PBy, PBz * PBz)) < fma(b.PAx, b.PAx, fma(b.PAy, b.PAy, b.PAz * b.PAz));
    const bool onD = fma(QDx, QDx, fma(QDy, QDy, QDz * QDz)) < fma(k.PAx, k.PAx, fma(k.PAy, k.PAy, k.PAz * k.PAz));
    const double AB = ax == 0 ? ABv[0] : (ax == 1 ? ABv[1] : ABv[2]);
    const double CD = ax == 0 ? CDv[0] : (ax == 1 ? CDv[1] : CDv[2]);
    const double pa = (ax == 0 ? b.PAx : (ax == 1 ? b.PAy : b.PAz)) + (onB ? AB : 0.0);   // P - (A or B)
    const double qc = (ax == 0 ? k.PAx : (ax == 1 ? k.PAy : k.PAz)) + (onD ? CD : 0.0);   // Q - (C or D)
    const double B00 = 0.5 * u * inv_s;
    const double B10 = b.inv2z * fma(-roz, u, 1.0);
    const double B01 = k.inv2z * fma(-roe, u, 1.0);
    const double C00 = fma(-roz * u, pq, pa);
    const double C01 = fma(roe * u, pq, qc);
    double g[NBR + 1][NKT + 1];
    g[0][0] = ax == 2 ? b.cc * k.cc * rs * w : 1.0;
#pragma unroll
    for (int n = 0; n < NBR; ++n) {
        double v = C00 * g[n][0];
        if (n > 0) v = fma((double)n * B10, g[n - 1][0], v);
        g[n + 1][0] = v;
    }
#pragma unroll
    for (int m = 0; m < NKT; ++m) {
#pragma unroll
        for (int n = 0; n <= NBR; ++n) {
            double v = C01 * g[n][m];
            if (m > 0) v = fma((double)m * B01, g[n][m - 1], v);
            if (n > 0) v = fma((double)n * B00, g[n - 1][m], v);
            g[n][m + 1] = v;
        }
    }
    // ket transfer (k on C, l on D), then bra transfer (i on A, j on B); from the near centre towards the far one:
    //   built on C: (k, l+1) = (k+1, l) + (C-D)(k, l)        built on D: (k+1, l) = (k, l+1) + (D-C)(k, l)
    double kt[NBR + 1][C::NKL];
#pragma unroll
    for (int n = 0; n <= NBR; ++n) {
        double h[NKT + 1];
#pragma unroll
        for (int m = 0; m <= NKT; ++m) h[m] = g[n][m];
        if (!onD) {
#pragma unroll
            for (int l = 0; l <= C::LD; ++l) {
#pragma unroll
                for (int kk = 0; kk <= C::LC; ++kk) kt[n][kk * (C::LD + 1) + l] = h[kk];
                if (l < C::LD) {
#pragma unroll
                    for (int m = 0; m < NKT - l; ++m) h[m] = fma(CD, h[m], h[m + 1]);
                }
            }
        } else {
#pragma unroll
            for (int kk = 0; kk <= C::LC; ++kk) {
#pragma unroll
                for (int l = 0; l <= C::LD; ++l) kt[n][kk * (C::LD + 1) + l] = h[l];
                if (kk < C::LC) {
#pragma unroll
                    for (int m = 0; m < NKT - kk; ++m) h[m] = fma(-CD, h[m], h[m + 1]);
                }
            }
        }
    }
#pragma unroll
    for (int kl = 0; kl < C::NKL; ++kl) {
        double f[NBR + 1];
#pragma unroll
        for (int n = 0; n <= NBR; ++n) f[n] = kt[n][kl];
        if (!onB) {
#pragma unroll
            for (int j = 0; j <= C::LB; ++j) {
#pragma unroll
                for (int i = 0; i <= C::LA; ++i) out[(i * (C::LB + 1) + j) * C::PADCD + kl] = f[i];
                if (j < C::LB) {
#pragma unroll
                    for (int n = 0; n < NBR - j; ++n) f[n] = fma(AB, f[n], f[n + 1]);
                }
            }
        } else {
#pragma unroll
            for (int i = 0; i <= C::LA; ++i) {
#pragma unroll
                for (int j = 0; j <= C::LB; ++j) out[(i * (C::LB + 1) + j) * C::PADCD + kl] = f[j];
                if (i < C::LA) {
#pragma unroll
                    for (int n = 0; n < NBR - i; ++n) f[n] = fma(-AB, f[n], f[n + 1]);
                }
            }
        }
    }
}

// phase 2 for the threads of cd chunk CHK: acc[n] += Gx*Gy*Gz over the nb items of the batch.
// The n-th integral of the chunk is the cd component pair q = CHK*CH + n = ic*ND + id (compile-time constants).
template <class C, int CHK, int n>
__device__ __forceinline__ void rys_fma_one(const double (&X)[C::NKL], const double (&Y)[C::NKL], const double (&Z)[C::NKL],
                                            double (&acc)[C::CH])
{
    constexpr int q = CHK * C::CH + n;
    if constexpr (q < C::NCD) {
        constexpr int ic = q / C::ND, id = q % C::ND;
        constexpr int ix = rys_cart(C::LC, ic, 0) * (C::LD + 1) + rys_cart(C::LD, id, 0);
        constexpr int iy = rys_cart(C::LC, ic, 1) * (C::LD + 1) + rys_cart(C::LD, id, 1);
        constexpr int iz = rys_cart(C::LC, ic, 2) * (C::LD + 1) + rys_cart(C::LD, id, 2);
        acc[n] = fma(X[ix] * Y[iy], Z[iz], acc[n]);
    }
}
template <class C, int CHK, int... Ns>
__device__ __forceinline__ void rys_fma_all(const double (&X)[C::NKL], const double (&Y)[C::NKL], const double (&Z)[C::NKL],
                                            double (&acc)[C::CH], std::integer_sequence<int, Ns...>)
{
    (rys_fma_one<C, CHK, Ns>(X, Y, Z, acc), ...);
}
template <class C, int CHK>
__device__ __forceinline__ void rys_phase2(const double *__restrict__ sm, int nb, int offx, int offy, int offz,
                                           double (&acc)[C::CH])
{
    for (int it = 0; it < nb; ++it) {
        const double *gx = sm + it * C::ITEMSZ + offx;
        const double *gy = sm + it * C::ITEMSZ + C::AXSZ + offy;
        const double *gz = sm + it * C::ITEMSZ + 2 * C::AXSZ + offz;
        double X[C::NKL], Y[C::NKL], Z[C::NKL];
#pragma unroll
        for (int q = 0; q < C::NKL; ++q) { X[q] = gx[q]; Y[q] = gy[q]; Z[q] = gz[q]; }
        rys_fma_all<C, CHK>(X, Y, Z, acc, std::make_integer_sequence<int, C::CH>{});
    }
}
template <class C, int CHK = 0>
__device__ __forceinline__ void rys_phase2_dispatch(int chunk, const double *__restrict__ sm, int nb, int offx, int offy,
                                                    int offz, double (&acc)[C::CH])
{
    if (chunk == CHK) rys_phase2<C, CHK>(sm, nb, offx, offy, offz, acc);
    else if constexpr (CHK + 1 < C::NCHT) rys_phase2_dispatch<C, CHK + 1>(chunk, sm, nb, offx, offy, offz, acc);
}

// (a5) digestion of the integrals a thread owns: (ia ib | q), q = CHK*CH + n.  Same six updates as DigestJK; WJ / WK
// select the J-only and K-only instantiations (the skipped matrix costs no loads, FMAs or reductions).
template <class C, int CHK, bool WJ, bool WK>
struct RysDigest {
    double jab, kac[C::NC], kad[C::ND], kbc[C::NC], kbd[C::ND];
    const double *D;
    double *J;
    int N, ra, rb, c0, d0, lane;
    double dab2;                 // 2 w D_ab (0 on idle lanes)

    template <int n>
    __device__ __forceinline__ void one(const double (&acc)[C::CH])
    {
        constexpr int q = CHK * C::CH + n;
        if constexpr (q < C::NCD) {
            constexpr int ic = q / C::ND, id = q % C::ND;
            const double v = acc[n];
            if constexpr (WJ) {
                jab = fma(__ldg(D + (size_t)(c0 + ic) * N + d0 + id), v, jab);
                double t = dab2 * v;                                        // J_cd: the lanes of a warp share (ic, id)
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
                if (lane == 0) atomicAdd(J + (size_t)(c0 + ic) * N + d0 + id, t);
            }
            if constexpr (WK) {
                const double Dbd = __ldg(D + (size_t)rb * N + d0 + id), Dbc = __ldg(D + (size_t)rb * N + c0 + ic);
                const double Dad = __ldg(D + (size_t)ra * N + d0 + id), Dac = __ldg(D + (size_t)ra * N + c0 + ic);
                kac[ic] = fma(Dbd, v, kac[ic]);
                kad[id] = fma(Dbc, v, kad[id]);
                kbc[ic] = fma(Dad, v, kbc[ic]);
                kbd[id] = fma(Dac, v, kbd[id]);
            }
        }
    }
    template <int... Ns>
    __device__ __forceinline__ void all(const double (&acc)[C::CH], std::integer_sequence<int, Ns...>) { (one<Ns>(acc), ...); }

    static __host__ __device__ constexpr bool touches_c(int ic)
    {
        for (int n = 0; n < C::CH; ++n) { const int q = CHK * C::CH + n; if (q < C::NCD && q / C::ND == ic) return true; }
        return false;
    }
    static __host__ __device__ constexpr bool touches_d(int id)
    {
        for (int n = 0; n < C::CH; ++n) { const int q = CHK * C::CH + n; if (q < C::NCD && q % C::ND == id) return true; }
        return false;
    }
    template <int ic>
    __device__ __forceinline__ void flush_c(double *K, double w)
    {
        if constexpr (touches_c(ic)) {
            atomicAdd(K + (size_t)ra * N + c0 + ic, w * kac[ic]);
            atomicAdd(K + (size_t)rb * N + c0 + ic, w * kbc[ic]);
        }
    }
    template <int id>
    __device__ __forceinline__ void flush_d(double *K, double w)
    {
        if constexpr (touches_d(id)) {
            atomicAdd(K + (size_t)ra * N + d0 + id, w * kad[id]);
            atomicAdd(K + (size_t)rb * N + d0 + id, w * kbd[id]);
        }
    }
    template <int... Is>
    __device__ __forceinline__ void flush_cs(double *K, double w, std::integer_sequence<int, Is...>) { (flush_c<Is>(K, w), ...); }
    template <int... Is>
    __device__ __forceinline__ void flush_ds(double *K, double w, std::integer_sequence<int, Is...>) { (flush_d<Is>(K, w), ...); }

    __device__ __forceinline__ void run(const double (&acc)[C::CH], bool active, int ia, int ib, const JKParams &p, int a0,
                                        int b0, int c0_, int d0_, double wgt, int lane_)
    {
        D = p.D; J = p.J; N = p.N; ra = a0 + ia; rb = b0 + ib; c0 = c0_; d0 = d0_; lane = lane_;
        const double w = active ? wgt : 0.0;
        dab2 = WJ ? (w + w) * __ldg(D + (size_t)ra * N + rb) : 0.0;
        jab = 0.0;
#pragma unroll
        for (int x = 0; x < C::NC; ++x) kac[x] = kbc[x] = 0.0;
#pragma unroll
        for (int x = 0; x < C::ND; ++x) kad[x] = kbd[x] = 0.0;
        all(acc, std::make_integer_sequence<int, C::CH>{});
        if (active) {
            if constexpr (WJ) atomicAdd(J + (size_t)ra * N + rb, (w + w) * jab);
            if constexpr (WK) {
                flush_cs(p.K, w, std::make_integer_sequence<int, C::NC>{});
                flush_ds(p.K, w, std::make_integer_sequence<int, C::ND>{});
            }
        }
    }
};
template <class C, bool WJ, bool WK, int CHK = 0>
__device__ __forceinline__ void rys_digest_dispatch(int chunk, const double (&acc)[C::CH], bool active, int ia, int ib,
                                                    const JKParams &p, int a0, int b0, int c0, int d0, double wgt, int lane)
{
    if (chunk == CHK) { RysDigest<C, CHK, WJ, WK> dg; dg.run(acc, active, ia, ib, p, a0, b0, c0, d0, wgt, lane); }
    else if constexpr (CHK + 1 < C::NCHT) rys_digest_dispatch<C, WJ, WK, CHK + 1>(chunk, acc, active, ia, ib, p, a0, b0, c0, d0, wgt, lane);
}

// contracted integrals of one shell quartet into the registers of the block (both phases, all batches)
template <class C>
__device__ __forceinline__ void rys_quartet(const PairTable &t, const RysTable &rt, double *__restrict__ sm, int bra_prim,
                                            int bra_stride, int bra_K, int ket_prim, int ket_stride, int ket_K,
                                            const double (&AB)[3], const double (&CD)[3], int chunk, int offx, int offy,
                                            int offz, double (&acc)[C::CH])
{
#pragma unroll
    for (int n = 0; n < C::CH; ++n) acc[n] = 0.0;
    const int nitems = bra_K * ket_K * C::NR;
    for (int base = 0; base < nitems; base += C::BATCH) {
        const int nb = nitems - base < C::BATCH ? nitems - base : C::BATCH;
        for (int unit = threadIdx.x; unit < 3 * nb; unit += C::NT) {
            const int it = unit / 3, ax = unit - 3 * it;
            const int item = base + it;
            const int pq = item / C::NR, r = item - pq * C::NR;
            const int kb = pq / ket_K, kk = pq - kb * ket_K;
            const PrimPair bp = load_prim(t, bra_prim + kb * bra_stride);
            const PrimPair kp = load_prim(t, ket_prim + kk * ket_stride);
            rys_phase1<C>(rt, bp, kp, r, ax, AB, CD, sm + it * C::ITEMSZ + ax * C::AXSZ);
        }
        __syncthreads();
        rys_phase2_dispatch<C>(chunk, sm, nb, offx, offy, offz, acc);
        __syncthreads();
    }
}

template <class C, bool WJ, bool WK>
__global__ void __launch_bounds__(C::NT, C::MINB) jk_rys_kernel(const JKParams p, const RysTable rt, unsigned long long *tile_counter)
{
    extern __shared__ double sm[];
    __shared__ long long s_tile;
    const int tid = threadIdx.x, lane = tid & 31;
    const int group = tid / C::NABP, ab = tid - group * C::NABP;
    const bool active = ab < C::NAB;
    const int ia = active ? ab / C::NB : 0, ib = active ? ab % C::NB : 0;
    const int offx = (rys_cart_rt<C::LA>(ia, 0) * (C::LB + 1) + rys_cart_rt<C::LB>(ib, 0)) * C::PADCD;
    const int offy = (rys_cart_rt<C::LA>(ia, 1) * (C::LB + 1) + rys_cart_rt<C::LB>(ib, 1)) * C::PADCD;
    const int offz = (rys_cart_rt<C::LA>(ia, 2) * (C::LB + 1) + rys_cart_rt<C::LB>(ib, 2)) * C::PADCD;
    unsigned long long cnt_q = 0ull, cnt_p = 0ull, cnt_n = 0ull;
    for (;;) {
        if (tid == 0) s_tile = (long long)atomicAdd(tile_counter, 1ull);
        __syncthreads();
        const long long w = s_tile * p.shard_count + p.shard_rank;
        __syncthreads();
        if (w >= p.total_warps) break;
        const int lo = find_segment(p, w);
        const Segment sg = p.segs[lo];
        const long long r = w - sg.warp_begin;
        const int i_base = sg.row_begin + (int)(r / sg.tiles_per_row) * TILE_R, j_base = ((int)(r % sg.tiles_per_row) + sg.col_tile_begin) * TILE_C;
        for (int jj = 0; jj < 32; ++jj) {                       // the 32 quartets of the tile, one after the other
            const int i = i_base + jj / TILE_C, j = j_base + (jj & (TILE_C - 1));
            if (i >= sg.rows) break;
            if (j >= (sg.same ? (i + 1) : sg.ket_n)) continue;
            const int gab = sg.bra_pair_base + i, gcd = sg.ket_pair_base + j;
            // the screen (DESIGN R-7; block-density rule R-23 when p.Dsh is set)
            const double S = (__ldg(p.t.Q + gab) * __ldg(p.t.Q + gcd)) * screen_density(p, gab, gcd);
            if (!(S >= p.tau && S < p.tau_hi)) continue;
            if (tid == 0) {
                cnt_q += 1ull;
                cnt_p += (unsigned long long)(sg.bra_K * sg.ket_K);
                cnt_n += (unsigned long long)((unsigned)__ldg(p.t.knom + gab) * (unsigned)__ldg(p.t.knom + gcd));
            }
            const int a0 = __ldg(p.t.bfa + gab), b0 = __ldg(p.t.bfb + gab);
            const double AB[3] = {__ldg(p.t.ABx + gab), __ldg(p.t.ABy + gab), __ldg(p.t.ABz + gab)};
            const double CD[3] = {__ldg(p.t.ABx + gcd), __ldg(p.t.ABy + gcd), __ldg(p.t.ABz + gcd)};
            const int sa = __ldg(p.t.sha + gab), sb = __ldg(p.t.shb + gab);
            const int sc = __ldg(p.t.sha + gcd), sd = __ldg(p.t.shb + gcd);
            double wgt = 1.0;
            if (sa == sb) wgt *= 0.5;
            if (sc == sd) wgt *= 0.5;
            if (gab == gcd) wgt *= 0.5;
            for (int ps = 0; ps < C::NPASS; ++ps) {
                const int chunk = ps * C::NCH + group;
                double acc[C::CH];
                rys_quartet<C>(p.t, rt, sm, sg.bra_prim_base + i, sg.bra_n, sg.bra_K, sg.ket_prim_base + j, sg.ket_n, sg.ket_K,
                               AB, CD, chunk, offx, offy, offz, acc);
                rys_digest_dispatch<C, WJ, WK>(chunk, acc, active, ia, ib, p, a0, b0, __ldg(p.t.bfa + gcd), __ldg(p.t.bfb + gcd), wgt, lane);
            }
        }
    }
    if (tid == 0 && cnt_q) {
        atomicAdd(p.counters, cnt_q);
        atomicAdd(p.counters + 1, cnt_p);
        atomicAdd(p.counters + 2, cnt_n);
    }
}

// (a2) Schwarz bound of the pairs of one sublist of class (la lb): the block evaluates (ab|ab) and takes the largest
// diagonal element |(mu nu|mu nu)|.  C must be RysCfg<la, lb, la, lb, NCH>.
template <class C, int CHK = 0>
__device__ __forceinline__ double rys_diag_max(int chunk, int ab, const double (&acc)[C::CH])
{
    double m = 0.0;
    if (chunk == CHK) {
#pragma unroll
        for (int n = 0; n < C::CH; ++n)
            if (CHK * C::CH + n == ab) m = fabs(acc[n]);
    } else if constexpr (CHK + 1 < C::NCHT) {
        m = rys_diag_max<C, CHK + 1>(chunk, ab, acc);
    }
    return m;
}

template <class C>
__global__ void __launch_bounds__(C::NT) schwarz_rys_kernel(const PairTable t, const RysTable rt, int pair_base, int prim_base,
                                                              int n, int K, double *__restrict__ Qout)
{
    extern __shared__ double sm[];
    __shared__ unsigned long long s_max;
    const int tid = threadIdx.x;
    const int group = tid / C::NABP, ab = tid - group * C::NABP;
    const bool active = ab < C::NAB;
    const int ia = active ? ab / C::NB : 0, ib = active ? ab % C::NB : 0;
    const int offx = (rys_cart_rt<C::LA>(ia, 0) * (C::LB + 1) + rys_cart_rt<C::LB>(ib, 0)) * C::PADCD;
    const int offy = (rys_cart_rt<C::LA>(ia, 1) * (C::LB + 1) + rys_cart_rt<C::LB>(ib, 1)) * C::PADCD;
    const int offz = (rys_cart_rt<C::LA>(ia, 2) * (C::LB + 1) + rys_cart_rt<C::LB>(ib, 2)) * C::PADCD;
    for (int j = blockIdx.x; j < n; j += gridDim.x) {
        const int g = pair_base + j;
        if (tid == 0) s_max = 0ull;
        const double AB[3] = {__ldg(t.ABx + g), __ldg(t.ABy + g), __ldg(t.ABz + g)};
        __syncthreads();                         // s_max is zero before any thread publishes its maximum
        for (int ps = 0; ps < C::NPASS; ++ps) {
            const int chunk = ps * C::NCH + group;
            double acc[C::CH];
            rys_quartet<C>(t, rt, sm, prim_base + j, n, K, prim_base + j, n, K, AB, AB, chunk, offx, offy, offz, acc);
            const double m = active ? rys_diag_max<C>(chunk, ab, acc) : 0.0;
            if (m > 0.0) atomicMax(&s_max, (unsigned long long)__double_as_longlong(m));
        }
        __syncthreads();
        if (tid == 0) Qout[g] = sqrt(__longlong_as_double((long long)s_max));
        __syncthreads();
    }
}

template <class C, bool WJ, bool WK>
inline cudaError_t launch_jk_rys(const JKParams &p, const RysTable &rt, unsigned long long *tile_counter, int nblocks, cudaStream_t st)
{
    auto kern = jk_rys_kernel<C, WJ, WK>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(tile_counter, 0, sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    kern<<<nblocks, C::NT, C::SMEM_BYTES, st>>>(p, rt, tile_counter);
    return cudaGetLastError();
}
template <class C>
inline cudaError_t launch_schwarz_rys(const PairTable &t, const RysTable &rt, int pair_base, int prim_base, int n, int K,
                                      double *Qout, int nblocks, cudaStream_t st)
{
    auto kern = schwarz_rys_kernel<C>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    kern<<<n < nblocks ? n : nblocks, C::NT, C::SMEM_BYTES, st>>>(t, rt, pair_base, prim_base, n, K, Qout);
    return cudaGetLastError();
}

}  // namespace adft
