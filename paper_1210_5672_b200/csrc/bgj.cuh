// bgj.cuh -- blocked Gauss-Jordan inverse of one 64 x 64 Schur block S = I/2 + kappa of the block LU (lu.cu; step S2,
// "LU-factorization"), for a CTA of 352 threads: eight warps apply rank-8 updates on the FP64 tensor pipe
// (DMMA.8x8x4), one warp inverts the 8 x 8 pivot blocks (roles: bgj_role).  Product code; shares nothing with oracle/.
//
// Panels of 8 pivots, p = 0..7, P = rows / columns 8p..8p+7, in place on W (starts as kappa, ends as F = inv(S) - 2 I):
//     D = I/2 + W_PP,  Dinv = inv(D) = 2 I + F_PP              (inverter warp: Neumann series on the tensor pipe, or elimination)
//     rows i not in P :  C' = W_iP Dinv = 2 W_iP + W_iP F_PP ;  W_ij -= C' W_Pj  (j not in P) ;  W_iP = -C'
//     rows P          :  W_Pj = Dinv W_Pj = 2 W_Pj + F_PP W_Pj  (j not in P) ;  W_PP = F_PP
// The diagonal is carried as a DEVIATION (kappa_jj = S_jj - 1/2 before its pivot, Z_jj - 2 after): the update formulas never
// touch the nominal part, so every entry of F keeps full relative accuracy.
// Warp w owns rows 8w..8w+7 as eight DMMA accumulator tiles (lane (fr, fk): row fr, columns 2 fk, 2 fk + 1 of each tile).
// The accumulator layout IS a valid A-operand layout when the contraction index is permuted (k-step s of lane fk stands for
// k = 2 fk + s); the B operands come from shared memory and are read with the same permutation -- no register shuffles.
// Look-ahead: after the barrier of panel p, warp p+1 updates its diagonal tile first and hands it to the inverter, which inverts
// it while the other warps finish the rank-8 update; one CTA-wide barrier per panel.
#pragma once
#include "common.cuh"

namespace sww {

// Warp roles.  A warp runs on scheduler (warp id mod 4), and a scheduler's DMMA pipe takes one DMMA per 16 cycles: the inverter's
// chain of dependent DMMAs must not queue behind the bulk updates, so warp 0 (the inverter) has scheduler 0 to itself --
// warps 4 and 8 idle through the inversion -- and the eight update warps are 1, 2, 3, 5, 6, 7, 9, 10 (schedulers 1, 2, 3).
constexpr int BGJ_CTA_THREADS = 352;   // threads of the calling CTA (11 warps)
constexpr int BGJ_THREADS = 288;       // threads that take part in the inversion (9 warps)
__device__ __forceinline__ int bgj_role(int warp) {  // 0..7: update warp owning that row block; 8: inverter; -1: idle
    if (warp == 0) return 8;
    if ((warp & 3) == 0 || warp > 10) return -1;
    return warp - 1 - (warp >> 2);
}
constexpr int BGJ_TLD = 66;   // leading dimension of the input tile T (row-major; even: entry pairs are 16-byte aligned)
constexpr int BGJ_RLD = 66;   // leading dimension of the pivot-row panel (8 x 64, row-major): conflict-free B-fragment loads
constexpr int BGJ_FLD = 10;   // leading dimension of the 8 x 8 pivot-block inverse
constexpr int BGJ_SCRATCH = 2 * 8 * BGJ_RLD + 2 * 8 * BGJ_FLD + 64;  // doubles: Rs[2], Fs8[2], Ds
constexpr double BGJ_PIVOT_GUARD = 1e-3;

__device__ __forceinline__ void bgj_dmma(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
__device__ __forceinline__ void bgj_bar_sync(int id, int n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void bgj_bar_arrive(int id, int n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }
constexpr int BGJ_BAR_FULL = 1, BGJ_BAR_TILE = 2, BGJ_BAR_TREAD = 3;

// reciprocal of a 2 x 2 pivot determinant (|d| ~ 1/4): MUFU seed (2^-20) + one cubic step r (1 + e + e^2), e = 1 - d r: 2^-60
__device__ __forceinline__ double bgj_rcp(double d) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
    const double e = fma(-d, r, 1.0);
    const double t = fma(e, e, e);
    return fma(r, t, r);
}

// One Gauss-Jordan step with a 2 x 2 pivot block (pivots 2 M, 2 M + 1) on the 8 x 8 block held by a warp, lane (r, q):
// a0 = W[r][2q], a1 = W[r][2q+1], diagonal in deviation form (S_jj - 1/2 before its pivot, Z_jj - 2 after).
// With D = [[a, b], [c, d]] (full values), det = a d - b c, inv(D) = adj(D) / det, everything that does not need 1/det is
// formed while the reciprocal is in flight; one multiply-add follows it:
//     rows not in the pair, columns not in the pair :  W -= (x adj(D) y) / det      x = my row at the pivot columns,
//     pivot rows, other columns                     :  W  = (adj(D) y) / det        y = the pivot rows at my column
//     other rows, pivot columns                     :  W  = -(x adj(D)) / det
//     pivot block                                   :  inv(D) - 2 I, with  d/det - 2 = (2 b c - 2 kappa_a d) / det  (no cancellation)
template <int M>
__device__ __forceinline__ void bgj_inv8_pair(double& a0, double& a1, int r, int q, double& dmin) {
    const unsigned full = 0xffffffffu;
    constexpr int R0 = 2 * M, R1 = 2 * M + 1;
    const double ka = __shfl_sync(full, a0, R0 * 4 + M), b = __shfl_sync(full, a1, R0 * 4 + M);   // pivot block (deviations on the diagonal)
    const double c = __shfl_sync(full, a0, R1 * 4 + M), kd = __shfl_sync(full, a1, R1 * 4 + M);
    const double x0 = __shfl_sync(full, a0, r * 4 + M), x1 = __shfl_sync(full, a1, r * 4 + M);    // my row at the pivot columns
    const double y00 = __shfl_sync(full, a0, R0 * 4 + q), y01 = __shfl_sync(full, a1, R0 * 4 + q);  // pivot rows at my columns
    const double y10 = __shfl_sync(full, a0, R1 * 4 + q), y11 = __shfl_sync(full, a1, R1 * 4 + q);
    const double a = 0.5 + ka, d = 0.5 + kd;
    const double bc = b * c;
    const double det = fma(a, d, -bc);
    const double rdet = bgj_rcp(det);
    dmin = fmin(dmin, fabs(det));
    // one branch-free path for all four cases: the pivot rows use x = -e_row and base 0 (W = adj(D) y / det), the pivot columns
    // use y = identity and base 0 (W = -(x adj(D)) / det); the four entries of the pivot block itself are patched at the end
    const bool prow = (r >> 1) == M, pcol = (q == M);
    const double xe0 = prow ? ((r == R0) ? -1.0 : 0.0) : x0, xe1 = prow ? ((r == R0) ? 0.0 : -1.0) : x1;
    const double z00 = pcol ? 1.0 : y00, z10 = pcol ? 0.0 : y10, z01 = pcol ? 0.0 : y01, z11 = pcol ? 1.0 : y11;
    const double base0 = (prow || pcol) ? 0.0 : a0, base1 = (prow || pcol) ? 0.0 : a1;
    const double w00 = fma(d, z00, -b * z10), w10 = fma(a, z10, -c * z00);   // adj(D) y, column 2q
    const double w01 = fma(d, z01, -b * z11), w11 = fma(a, z11, -c * z01);   // column 2q + 1
    const double s0 = fma(xe0, w00, xe1 * w10), s1 = fma(xe0, w01, xe1 * w11);
    const double two_bc = 2.0 * bc;
    const double f00 = fma(-2.0 * ka, d, two_bc), f11 = fma(-2.0 * kd, a, two_bc);  // (inv(D) - 2 I) det on the diagonal
    double v0 = fma(-s0, rdet, base0), v1 = fma(-s1, rdet, base1);
    if (prow && pcol) {
        if (r == R0) v0 = f00 * rdet;
        else v1 = f11 * rdet;
    }
    a0 = v0;
    a1 = v1;
}

// inv(D) - 2 I of an 8 x 8 pivot block D = I/2 + kappa = (I - x)/2, x = -2 kappa, by the Neumann series in product form on the
// tensor pipe:  inv(I - x) = (I + x)(I + x^2)(I + x^4)...,  carried as the deviation y = inv(I - x) - I:
//     y <- y + x^(2^l) + y x^(2^l),  l = 1..L ;   inv(D) - 2 I = 2 y ;   truncation |x|^(2^(L+1)).
// A scalar elimination is a chain of 8 dependent reciprocals (~1300 cycles for one warp); this is L + 1 dependent 8 x 8 products
// (~300 cycles).  Every matrix is kept with its transpose, both in accumulator layout: the accumulator layout of M is an
// A operand and that of M^T is a B operand of DMMA.8x8x4 under the same permuted contraction index (no shuffles), and all
// factors are polynomials in x, so (p q)^T = p^T q^T.
// Applicable when 8 max|x_ij| <= 0.3 (then L = 3 or 4 gives |x|^(2^(L+1)) < 1e-16); returns false otherwise (warp-uniform) and the
// caller eliminates instead.  Second-kind kernels have kappa_ij = O(1/N): the bound is 0.014 at the metric point.
__device__ __forceinline__ bool bgj_inv8_neumann(const double* Ds, int fr, int fk, double& f0, double& f1) {
    const double2 xr = *reinterpret_cast<const double2*>(Ds + fr * 8 + 2 * fk);
    const double x0 = -2.0 * xr.x, x1 = -2.0 * xr.y;                                              // x   in accumulator layout
    const double t0 = -2.0 * Ds[(2 * fk) * 8 + fr], t1 = -2.0 * Ds[(2 * fk + 1) * 8 + fr];      // x^T in accumulator layout
    // An 8 x 8 product P Q in accumulator layout is two chained DMMAs, dmma(A = P.k0, B = Q^T.k0) then (P.k1, Q^T.k1); one warp
    // issues in order, so the k-steps of independent products are interleaved by hand (a dependent DMMA waits 26 cycles).
    double s0 = 0.0, s1 = 0.0, u0 = 0.0, u1 = 0.0;       // s = x^2, u = (x^2)^T
    bgj_dmma(s0, s1, x0, t0);
    bgj_dmma(u0, u1, t0, x0);
    bgj_dmma(s0, s1, x1, t1);
    bgj_dmma(u0, u1, t1, x1);
    // max |x_ij| over the block (the high words of non-negative doubles order like the doubles); the reduction is in flight
    // while the series runs and is looked at afterwards
    const unsigned hi = (unsigned)__double2hiint(fmax(fabs(x0), fabs(x1)));
    const double bound = 8.0 * __hiloint2double((int)__reduce_max_sync(0xffffffffu, hi), -1);
    double y0 = x0, y1 = x1;
    auto level = [&](bool squares) {
        double n0 = 0.0, n1 = 0.0, v0 = 0.0, v1 = 0.0;   // the next squares head the dependent chain
        double c0 = y0 + s0, c1 = y1 + s1;               // y + x^(2^l) + y x^(2^l)
        if (squares) {
            bgj_dmma(n0, n1, s0, u0);
            bgj_dmma(v0, v1, u0, s0);
        }
        bgj_dmma(c0, c1, y0, u0);
        if (squares) {
            bgj_dmma(n0, n1, s1, u1);
            bgj_dmma(v0, v1, u1, s1);
        }
        bgj_dmma(c0, c1, y1, u1);
        y0 = c0; y1 = c1;
        s0 = n0; s1 = n1; u0 = v0; u1 = v1;
    };
    level(true);    // through x^3
    level(true);    // through x^7
    if (bound <= 0.1) {
        level(false);   // through x^15
    } else {
        level(true);
        level(false);   // through x^31
    }
    f0 = 2.0 * y0;
    f1 = 2.0 * y1;
    return bound <= 0.3;
}

// the work of one update warp for panel P (after the barrier that made F_PP and the pivot-row panel visible)
template <int P>
__device__ __forceinline__ void bgj_panel(double (&acc)[8][2], int w, int fr, int fk, double* Rs, const double* Fs8, double* Ds) {
    const double* R = Rs + (P & 1) * 8 * BGJ_RLD;
    const double* F8 = Fs8 + (P & 1) * 8 * BGJ_FLD;
    // B fragments with the permuted contraction index: k-step s of lane fk is k = 2 fk + s
    auto rb = [&](int t, int s) { return R[(2 * fk + s) * BGJ_RLD + 8 * t + fr]; };
    auto write_row = [&](double* dst) {  // my 8 x 64 row block -> dst[k = fr][n]
#pragma unroll
        for (int t = 0; t < 8; t++) *reinterpret_cast<double2*>(dst + fr * BGJ_RLD + 8 * t + 2 * fk) = make_double2(acc[t][0], acc[t][1]);
    };
    if (w != P) {
        // C' = 2 C + C F_PP  (A = C in accumulator layout, B = F_PP[k][n = fr])
        double c0 = 2.0 * acc[P][0], c1 = 2.0 * acc[P][1];
        bgj_dmma(c0, c1, acc[P][0], F8[(2 * fk) * BGJ_FLD + fr]);
        bgj_dmma(c0, c1, acc[P][1], F8[(2 * fk + 1) * BGJ_FLD + fr]);
        const double n0 = -c0, n1 = -c1;
        constexpr int PN = (P + 1) & 7;
        const bool next_owner = (P < 7) && (w == P + 1);
        if (next_owner) {  // look-ahead: the next pivot block first, handed to the inverter at once
            bgj_dmma(acc[PN][0], acc[PN][1], n0, rb(PN, 0));
            bgj_dmma(acc[PN][0], acc[PN][1], n1, rb(PN, 1));
            *reinterpret_cast<double2*>(Ds + fr * 8 + 2 * fk) = make_double2(acc[PN][0], acc[PN][1]);
            bgj_bar_arrive(BGJ_BAR_TILE, 64);
        }
#pragma unroll
        for (int s = 0; s < 2; s++)   // the two k-steps of a tile depend on each other: all first steps, then all second steps
#pragma unroll
            for (int t = 0; t < 8; t++) {
                if (t == P || (next_owner && t == PN)) continue;
                bgj_dmma(acc[t][0], acc[t][1], s ? n1 : n0, rb(t, s));
            }
        acc[P][0] = n0;
        acc[P][1] = n1;
        if (next_owner) write_row(Rs + (PN & 1) * 8 * BGJ_RLD);
    } else {
        // rows P: W_Pj = 2 W_Pj + F_PP W_Pj  (A = F_PP in accumulator layout, B = the raw row panel)
        const double2 fa = *reinterpret_cast<const double2*>(F8 + fr * BGJ_FLD + 2 * fk);
#pragma unroll
        for (int t = 0; t < 8; t++) {
            acc[t][0] *= 2.0;
            acc[t][1] *= 2.0;
        }
#pragma unroll
        for (int s = 0; s < 2; s++)
#pragma unroll
            for (int t = 0; t < 8; t++) {
                if (t == P) continue;
                bgj_dmma(acc[t][0], acc[t][1], s ? fa.y : fa.x, rb(t, s));
            }
        acc[P][0] = fa.x;
        acc[P][1] = fa.y;
    }
}

// T (shared, row-major, leading dimension BGJ_TLD, 16-byte aligned) holds kappa = S - I/2.  On return F = inv(S) - 2 I is in Fg (global, column-major,
// ld 64; skipped when Fg == nullptr) and in sF (shared, column-major, ld 68: the DMMA operand layout of lu.cu).  Every one of the 352 threads must call it;
// scr: BGJ_SCRATCH doubles of shared memory.  The two idle warps return as soon as every active warp has read T (from then on
// the caller may overwrite it); the active warps end with a barrier among themselves: the caller must follow with a CTA-wide
// barrier before anybody reads sF.
// hook(p) is called by every thread right after the barrier of panel p (the spine uses it to poll flags / issue prefetches).
template <class Hook>
__device__ __forceinline__ void bgj64(const double* T, double* scr, int* status, int tid, double* Fg, double* sF, Hook&& hook) {
    const int w = bgj_role(tid >> 5), lane = tid & 31, fr = lane >> 2, fk = lane & 3;
    if (w < 0) {  // idle warps: back to the caller as soon as T is in the registers of the others (the caller may reuse T)
        bgj_bar_sync(BGJ_BAR_TREAD, BGJ_CTA_THREADS);
        return;
    }
    double* Rs = scr;                        // [2][8][RLD]
    double* Fs8 = scr + 2 * 8 * BGJ_RLD;     // [2][8][FLD]
    double* Ds = Fs8 + 2 * 8 * BGJ_FLD;      // [8][8]
    if (w == 8) {
        // ------------------------------------------------------------------ the inverter
        bgj_bar_arrive(BGJ_BAR_TREAD, BGJ_CTA_THREADS);
        double pmin = 1.0;
#pragma unroll 1
        for (int p = 0; p < 8; p++) {
            bgj_bar_sync(BGJ_BAR_TILE, 64);  // Ds holds the pivot block of panel p
            double a0, a1;
            if (!bgj_inv8_neumann(Ds, fr, fk, a0, a1)) {  // a block that is not a small perturbation of I/2: eliminate
                a0 = Ds[fr * 8 + 2 * fk];
                a1 = Ds[fr * 8 + 2 * fk + 1];
                bgj_inv8_pair<0>(a0, a1, fr, fk, pmin);
                bgj_inv8_pair<1>(a0, a1, fr, fk, pmin);
                bgj_inv8_pair<2>(a0, a1, fr, fk, pmin);
                bgj_inv8_pair<3>(a0, a1, fr, fk, pmin);
            }
            double* F8 = Fs8 + (p & 1) * 8 * BGJ_FLD;
            *reinterpret_cast<double2*>(F8 + fr * BGJ_FLD + 2 * fk) = make_double2(a0, a1);
            bgj_bar_sync(BGJ_BAR_FULL, BGJ_THREADS);
            hook(p);
        }
        if (lane == 0 && !(pmin >= BGJ_PIVOT_GUARD * BGJ_PIVOT_GUARD)) atomicCAS(status, SWW_OK, SWW_ESINGULAR);
        bgj_bar_sync(BGJ_BAR_FULL, BGJ_THREADS);  // the closing barrier
        return;
    }
    // ---------------------------------------------------------------------- the update warps
    double acc[8][2];
#pragma unroll
    for (int t = 0; t < 8; t++) {
        const double2 tv = *reinterpret_cast<const double2*>(T + (8 * w + fr) * BGJ_TLD + 8 * t + 2 * fk);
        acc[t][0] = tv.x;
        acc[t][1] = tv.y;
    }
    bgj_bar_arrive(BGJ_BAR_TREAD, BGJ_CTA_THREADS);
    if (w == 0) {
#pragma unroll
        for (int t = 0; t < 8; t++) *reinterpret_cast<double2*>(Rs + fr * BGJ_RLD + 8 * t + 2 * fk) = make_double2(acc[t][0], acc[t][1]);
        *reinterpret_cast<double2*>(Ds + fr * 8 + 2 * fk) = make_double2(acc[0][0], acc[0][1]);
        bgj_bar_arrive(BGJ_BAR_TILE, 64);
    }
#define SWW_BGJ_PANEL(P)                                                                             \
    bgj_bar_sync(BGJ_BAR_FULL, BGJ_THREADS); /* F_PP and the pivot-row panel are in shared memory */ \
    hook(P);                                                                                         \
    bgj_panel<P>(acc, w, fr, fk, Rs, Fs8, Ds);
    SWW_BGJ_PANEL(0) SWW_BGJ_PANEL(1) SWW_BGJ_PANEL(2) SWW_BGJ_PANEL(3)
    SWW_BGJ_PANEL(4) SWW_BGJ_PANEL(5) SWW_BGJ_PANEL(6) SWW_BGJ_PANEL(7)
#undef SWW_BGJ_PANEL
#pragma unroll
    for (int t = 0; t < 8; t++)
#pragma unroll
        for (int e = 0; e < 2; e++) {
            const int row = 8 * w + fr, col = 8 * t + 2 * fk + e;
            if (Fg) Fg[col * 64 + row] = acc[t][e];
            sF[col * 68 + row] = acc[t][e];
        }
    bgj_bar_sync(BGJ_BAR_FULL, BGJ_THREADS);  // the closing barrier
}

__device__ __forceinline__ void bgj64(const double* T, double* scr, int* status, int tid, double* Fg, double* sF) {
    bgj64(T, scr, status, tid, Fg, sF, [](int) {});
}

}  // namespace sww
