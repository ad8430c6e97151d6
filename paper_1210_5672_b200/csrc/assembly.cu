// assembly.cu -- steps S0 (node preparation) and S1 (kernel-matrix assembly) of the DtN setup.
//   S0: eta' = D eta, eta'' = D(D eta) by the Fourier differentiation circulant carried in double-double (R4, R8),
//       per-node tables exp(-(h+eta_j)) (image term) and, for the dd path, sinh/cosh(eta_j).
//   S1: K_ij, G_ij of (2.13) with the image kernels subtracted (R1; (A.2),(A.3),(A.8));
//       diagonal from the limits of PAPER.md:150, 653, 673.  Also writes A - I/2 = K (2.7) into the LU buffer (lu.cu keeps the 1/2 of the pivots implicit).
// Layout: K, G, LU column-major (entry (i,j) at i + j*N): a warp writes 32 consecutive i for one j (coalesced 256 B).
// Product code; shares nothing with oracle/.
#include "common.cuh"
#include "dd.cuh"

namespace sww {

// ------------------------------------------------------------------------------------------------ S0: node preparation
// exp / expm1 / sinh / cosh for the node tables with the series divisions replaced by dd reciprocals from a shared table
// rn[n] (+ rn[32 + n]) = 1 / n, n = 1..31 (one accurate division per lane instead of ~80 per node)
__device__ __forceinline__ dd exp_series_tab(dd r, const double* rn, bool minus_one) {
    dd term = minus_one ? r : dd{1.0, 0.0}, sum = term;
    for (int n = minus_one ? 2 : 1; n <= 27; n++) {
        term = dd_mul(dd_mul(term, r), dd{rn[n], rn[32 + n]});
        sum = dd_add(sum, term);
    }
    return sum;
}
__device__ __forceinline__ dd dd_exp_tab(dd x, const double* rn) {
    double kf = rint(x.hi * 1.4426950408889634074);
    dd r = dd_sub(x, dd_mul_d(dd_ln2(), kf));
    return dd_ldexp(exp_series_tab(r, rn, false), (int)kf);
}
__device__ __forceinline__ dd dd_expm1_tab(dd x, const double* rn) {
    if (fabs(x.hi) < 0.34) return exp_series_tab(x, rn, true);
    return dd_add_d(dd_exp_tab(x, rn), -1.0);
}
__device__ __forceinline__ void dd_sinhcosh_tab_n(dd x, const double* rn, dd* sh, dd* ch) {
    if (fabs(x.hi) < 0.5) {
        dd x2 = dd_sqr(x);
        dd ts = x, tc = dd{1.0, 0.0}, ss = x, cc = dd{1.0, 0.0};
        for (int n = 1; n <= 15; n++) {
            tc = dd_mul(dd_mul(dd_mul(tc, x2), dd{rn[2 * n - 1], rn[32 + 2 * n - 1]}), dd{rn[2 * n], rn[32 + 2 * n]});
            ts = dd_mul(dd_mul(dd_mul(ts, x2), dd{rn[2 * n], rn[32 + 2 * n]}), dd{rn[2 * n + 1], rn[32 + 2 * n + 1]});
            cc = dd_add(cc, tc);
            ss = dd_add(ss, ts);
        }
        *sh = ss;
        *ch = cc;
        return;
    }
    dd e = dd_exp_tab(x, rn);
    dd ei = dd_div(dd{1.0, 0.0}, e);
    *sh = dd_half(dd_sub(e, ei));
    *ch = dd_half(dd_add(e, ei));
}

// S0 in ONE launch.  Per node i (four warps per node, two nodes per CTA of 8 warps):
//   d1_i = sum_{m=1}^{N/2-1} dc[m] (f_{i-m} - f_{i+m}),  dc[m] = (1/2)(-1)^m cot(pi m/N)   (eta' = D eta; Nyquist symbol 0, R4)
//   d2_i = c2[0] f_i + sum_{m=1}^{N/2} c2[m] (f_{i-m} + f_{i+m})                             (eta'' = D(D eta) as one circulant:
//          symbol -k^2, 0 at the Nyquist mode; c2[N/2] is stored halved because the sum meets that node twice; tables.cu)
//   and the per-node tables in dd (planar): E = exp(-(h+eta)), Dm = 1 - E (via expm1) for the image term, sinh/cosh(eta) for the dd
//   kernels (the fp64 assembly reads the hi planes of E, Dm; the dd assembly and the dd base-state pass read everything).
// The sums are chains of dependent dd operations behind scattered loads (their time is the length of the per-lane chain: four
// independent chains per sum and lane); the three series of the tables run on lane 0 of the warps 1..3 of the node meanwhile.
// Until round 2 these were three launches (D, D again on its own output, the tables): at N = 256 a third of a stage's launches.
__global__ void __launch_bounds__(256) k_node_prep(int N, double h, int finite, const double* __restrict__ dc, const double* __restrict__ dc2,
                                                   const double* __restrict__ f, double* __restrict__ d1, double* __restrict__ d2,
                                                   double* __restrict__ E, double* __restrict__ Dm, double* __restrict__ Sh, double* __restrict__ Ch,
                                                   int* status) {
    __shared__ double part[2][4][4];
    __shared__ double rn[64];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, node = warp >> 2, q = warp & 3;
    const int i = blockIdx.x * 2 + node, mask = N - 1;
    const int l128 = q * 32 + lane;  // position among the 128 lanes that share the node
    if (threadIdx.x >= 1 && threadIdx.x < 32) {  // rn[n] (+ rn[32 + n]) = 1 / n for the series of the tables
        const dd r = dd_div(dd{1.0, 0.0}, dd{(double)threadIdx.x, 0.0});
        rn[threadIdx.x] = r.hi;
        rn[32 + threadIdx.x] = r.lo;
    }
    dd a1[4] = {{0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}};  // independent chains: a dd multiply-add is ~30 dependent instructions
    dd a2[4] = {{0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}};
    if (i < N) {
        if (l128 == 0) a2[0] = dd_mul(dd_load(dc2, N, 0), dd_load(f, N, i));
        for (int m0 = 1 + l128; m0 <= N / 2; m0 += 512) {
            dd c[4], e[4], a[4], b[4];
            bool on[4];
#pragma unroll
            for (int u = 0; u < 4; u++) {  // the loads of a group are issued together
                const int m = m0 + 128 * u;
                on[u] = m <= N / 2;        // dc[N/2] = 0, dc2[N/2] halved: the Nyquist node is met once, with both neighbours equal
                const int mm = on[u] ? m : 0;
                c[u] = dd_load(dc, N, mm);
                e[u] = dd_load(dc2, N, mm);
                a[u] = dd_load(f, N, (i - mm) & mask);
                b[u] = dd_load(f, N, (i + mm) & mask);
            }
#pragma unroll
            for (int u = 0; u < 4; u++)
                if (on[u]) {
                    a1[u] = dd_fma(c[u], dd_sub(a[u], b[u]), a1[u]);
                    a2[u] = dd_fma(e[u], dd_add(a[u], b[u]), a2[u]);
                }
        }
    }
    dd s1 = dd_warp_sum(dd_add(dd_add(a1[0], a1[1]), dd_add(a1[2], a1[3])));
    dd s2 = dd_warp_sum(dd_add(dd_add(a2[0], a2[1]), dd_add(a2[2], a2[3])));
    if (lane == 0) {
        part[node][q][0] = s1.hi; part[node][q][1] = s1.lo;
        part[node][q][2] = s2.hi; part[node][q][3] = s2.lo;
    }
    __syncthreads();  // the partial sums and rn
    if (lane != 0 || i >= N) return;
    if (q == 0) {
        for (int r = 1; r < 4; r++) {
            s1 = dd_add(s1, dd{part[node][r][0], part[node][r][1]});
            s2 = dd_add(s2, dd{part[node][r][2], part[node][r][3]});
        }
        dd_store(d1, N, i, s1);
        dd_store(d2, N, i, s2);
        return;
    }
    const dd e = dd_load(f, N, i);
    if (q == 3) {
        dd sh, ch;
        dd_sinhcosh_tab_n(e, rn, &sh, &ch);
        dd_store(Sh, N, i, sh);
        dd_store(Ch, N, i, ch);
    } else if (finite) {
        const dd Y = dd_add_d(e, h);
        if (q == 1) {
            if (!(Y.hi > 0.0)) atomicCAS(status, SWW_OK, SWW_EBOTTOM);
            dd_store(E, N, i, dd_exp_tab(dd_neg(Y), rn));
        } else {
            dd_store(Dm, N, i, dd_neg(dd_expm1_tab(dd_neg(Y), rn)));
        }
    }
}

// ------------------------------------------------------------------------------------------------ S1: fp64 assembly
// sinh(y), cosh(y) evaluated DIRECTLY from y = eta_i - eta_j (never from per-node tables: next to the diagonal the addition
// formulas lose N/(2 pi |i-j|) digits -- DESIGN.md section 5).  |y| <= 1: odd/even Taylor polynomials in y^2; else from exp.
__device__ __forceinline__ void sinhcosh_f64(double y, double* sh, double* ch) {
    double a = fabs(y);
    if (a <= 1.0) {
        double t = y * y;
        // sinh(y)/y = sum t^n/(2n+1)!, n = 0..10 ; cosh(y) = sum t^n/(2n)!, n = 0..10
        double ps = 1.9572941063391263e-20;  // 1/21!
        ps = fma(ps, t, 8.2206352466243295e-18);  // 1/19!
        ps = fma(ps, t, 2.8114572543455206e-15);  // 1/17!
        ps = fma(ps, t, 7.6471637318198164e-13);  // 1/15!
        ps = fma(ps, t, 1.6059043836821613e-10);  // 1/13!
        ps = fma(ps, t, 2.5052108385441720e-08);  // 1/11!
        ps = fma(ps, t, 2.7557319223985893e-06);  // 1/9!
        ps = fma(ps, t, 1.9841269841269841e-04);  // 1/7!
        ps = fma(ps, t, 8.3333333333333332e-03);  // 1/5!
        ps = fma(ps, t, 1.6666666666666666e-01);  // 1/3!
        *sh = fma(y * t, ps, y);
        double pc = 4.1103176233121648e-19;  // 1/20!
        pc = fma(pc, t, 1.5619206968586225e-16);  // 1/18!
        pc = fma(pc, t, 4.7794773323873853e-14);  // 1/16!
        pc = fma(pc, t, 1.1470745597729725e-11);  // 1/14!
        pc = fma(pc, t, 2.0876756987868100e-09);  // 1/12!
        pc = fma(pc, t, 2.7557319223985888e-07);  // 1/10!
        pc = fma(pc, t, 2.4801587301587302e-05);  // 1/8!
        pc = fma(pc, t, 1.3888888888888889e-03);  // 1/6!
        pc = fma(pc, t, 4.1666666666666664e-02);  // 1/4!
        pc = fma(pc, t, 0.5);
        *ch = fma(t, pc, 1.0);
    } else {
        double e = exp(a), ei = 1.0 / e;
        *ch = 0.5 * (e + ei);
        *sh = copysign(0.5 * (e - ei), y);
    }
}

constexpr int ASM_TI = 128;  // rows (targets i) per block = threads per block
constexpr int ASM_TJ = 32;   // columns (sources j) per block

// sin, cos of delta = p_i - p_j (p = xi - alpha) from the per-node double-double tables S = sin p, C = cos p: the difference
// S_i C_j - C_i S_j cancels next to the diagonal, so the products are taken exactly and the low words are carried -- the
// x-differences of a refined mesh are then as accurate as the exact tables of the uniform one.
__device__ __forceinline__ void mesh_delta(double Si, double Sil, double Ci, double Cil, double Sj, double Sjl, double Cj, double Cjl,
                                           double* sd, double* cd) {
    const double p = Ci * Sj, e = fma(Ci, Sj, -p);
    const double low = fma(Sil, Cj, Si * Cjl) - fma(Cil, Sj, Ci * Sjl);
    *sd = (fma(Si, Cj, -p) - e) + low;
    *cd = fma(Ci, Cj, Si * Sj);
}
// sin^2(x/2) from sin x, cos x without cancellation
__device__ __forceinline__ double half_angle_sq(double sx, double cx) { return cx >= 0.0 ? sx * sx / (2.0 * (1.0 + cx)) : 0.5 * (1.0 - cx); }

// MESH: the refined mesh x = xi(alpha) of (2.10) (mesh.cu): zeta' = xE + i d1, zeta'' = xE1 + i d2, Re(zeta_i - zeta_j) =
// (alpha_i - alpha_j) + (p_i - p_j); the regularizing cot((alpha_i - alpha_j)/2) of (2.13) keeps the uniform table.
template <bool FINITE, int TJ, bool MESH>
__global__ void __launch_bounds__(ASM_TI) k_assemble_f64(int N, const double* __restrict__ eta, const double* __restrict__ d1,
                                                         const double* __restrict__ d2, const double* __restrict__ E,
                                                         const double* __restrict__ Dm, const double* __restrict__ cs,
                                                         const double* __restrict__ sn, const double* __restrict__ c0,
                                                         const double* __restrict__ s2, MeshDev ms, double* __restrict__ K,
                                                         double* __restrict__ G, double* __restrict__ LU) {
    __shared__ double s_eta[TJ], s_d1[TJ], s_E[TJ], s_Dm[TJ];
    __shared__ double s_xE[MESH ? TJ : 1], s_xS[MESH ? 2 * TJ : 1], s_xC[MESH ? 2 * TJ : 1];
    __shared__ double s_cs[ASM_TI + TJ], s_sn[ASM_TI + TJ], s_c0[ASM_TI + TJ], s_s2[ASM_TI + TJ];
    const int tid = threadIdx.x, mask = N - 1;
    const int i0 = blockIdx.x * ASM_TI, j0 = blockIdx.y * TJ;
    if (tid < TJ) {
        int j = (j0 + tid) & mask;
        s_eta[tid] = eta[j];
        s_d1[tid] = d1[j];
        if (FINITE) {
            s_E[tid] = E[j];
            s_Dm[tid] = Dm[j];
        }
        if (MESH) {
            s_xE[tid] = ms.xE[j];
            s_xS[tid] = ms.xS[j]; s_xS[TJ + tid] = ms.xS[N + j];
            s_xC[tid] = ms.xC[j]; s_xC[TJ + tid] = ms.xC[N + j];
        }
    }
    // table slice: index s <-> m = (i0 - j0 - (TJ-1) + s) mod N, s = tid - jj + TJ - 1
    for (int s = tid; s < ASM_TI + TJ - 1; s += ASM_TI) {
        int m = (i0 - j0 - (TJ - 1) + s) & mask;
        s_cs[s] = cs[m];
        s_sn[s] = sn[m];
        s_c0[s] = c0[m];
        s_s2[s] = s2[m];
    }
    __syncthreads();
    const int i = i0 + tid;
    if (i >= N) return;
    const double eta_i = eta[i], d1_i = d1[i], d2_i = d2[i];
    const double E_i = FINITE ? E[i] : 0.0, Dm_i = FINITE ? Dm[i] : 0.0;
    const double rN = 1.0 / (double)N;
    const int jmax = min(TJ, N - j0);
    double xE_i = 1.0, xE1_i = 0.0, xS_i = 0.0, xSl_i = 0.0, xC_i = 1.0, xCl_i = 0.0;
    if (MESH) {
        xE_i = ms.xE[i]; xE1_i = ms.xE1[i];
        xS_i = ms.xS[i]; xSl_i = ms.xS[N + i];
        xC_i = ms.xC[i]; xCl_i = ms.xC[N + i];
    }
    for (int jj = 0; jj < jmax; jj++) {
        const int j = j0 + jj, s = tid - jj + TJ - 1;
        double sx = s_sn[s], cx = s_cs[s], sq = s_s2[s];
        const double d1_j = s_d1[jj], xE_j = MESH ? s_xE[jj] : 1.0;
        if (MESH) {
            double sd, cd;
            mesh_delta(xS_i, xSl_i, xC_i, xCl_i, s_xS[jj], s_xS[TJ + jj], s_xC[jj], s_xC[TJ + jj], &sd, &cd);
            const double s0 = sx, c0m = cx;
            sx = fma(s0, cd, c0m * sd);
            cx = fma(c0m, cd, -s0 * sd);
            sq = half_angle_sq(sx, cx);
        }
        double k1, g1;
        if (MESH && i != j) {
            double y = eta_i - s_eta[jj];
            double sh, ch;
            sinhcosh_f64(y, &sh, &ch);
            double p = (cx >= 0.0) ? (cx + ch) / fma(sx, sx, sh * sh) : 1.0 / (ch - cx);
            double hp = 0.5 * p;
            k1 = hp * fma(d1_j, sx, -xE_j * sh);                    // Im{ zeta'_j (1/2)cot }
            g1 = fma(hp, fma(d1_i, sh, xE_i * sx), -s_c0[s]);       // Re{ zeta'_i (1/2)cot } - (1/2)cot((alpha_i - alpha_j)/2)
        } else if (MESH) {
            double den = 2.0 * fma(d1_i, d1_i, xE_i * xE_i);
            k1 = -fma(d2_i, xE_i, -xE1_i * d1_i) / den;             // -Im{ zeta''/(2 zeta') }
            g1 = fma(xE1_i, xE_i, d1_i * d2_i) / den;               //  Re{ zeta''/(2 zeta') }
        } else if (i != j) {
            double y = eta_i - s_eta[jj];  // Im(zeta_i - zeta_j) from the raw inputs
            double sh, ch;
            sinhcosh_f64(y, &sh, &ch);
            // (1/2) cot((x+iy)/2) = (1/2) p (sin x - i sinh y), two-branch p of PAPER.md:154
            double p = (cx >= 0.0) ? (cx + ch) / fma(sx, sx, sh * sh) : 1.0 / (ch - cx);
            double hp = 0.5 * p;
            k1 = hp * fma(d1_j, sx, -sh);           // Im{ zeta'_j (1/2)cot }
            g1 = fma(hp, fma(d1_i, sh, sx), -s_c0[s]);  // Re{ zeta'_i (1/2)cot } - (1/2)cot(x/2)
        } else {
            double den = 2.0 * fma(d1_i, d1_i, 1.0);
            k1 = -d2_i / den;        // -Im{ zeta''/(2 zeta') }
            g1 = d1_i * d2_i / den;  //  Re{ zeta''/(2 zeta') }
        }
        double k2 = 0.0, g2 = 0.0;
        if (FINITE) {
            // image point: (1/2)cot((x + i y2)/2), y2 = Y_i + Y_j > 0, written with Eij = exp(-y2) = E_i E_j:
            //   c_r = Eij sin x / den, c_i = -(1 - Eij^2) / (2 den), den = (1 - Eij)^2 + 4 Eij sin^2(x/2)   (all terms positive)
            double Eij = E_i * s_E[jj];
            double omE = fma(E_i, s_Dm[jj], Dm_i);  // 1 - E_i E_j = Dm_i + E_i Dm_j
            double den = fma(omE, omE, 4.0 * Eij * sq);
            double inv = 1.0 / den;
            double cr = Eij * sx * inv;
            double ci = -0.5 * omE * (1.0 + Eij) * inv;
            k2 = MESH ? fma(-d1_j, cr, xE_j * ci) : fma(-d1_j, cr, ci);  // Im{ conj(zeta'_j) (1/2)cot }
            g2 = MESH ? fma(-d1_i, ci, xE_i * cr) : fma(-d1_i, ci, cr);  // Re{ zeta'_i (1/2)cot }
        }
        double kv = (k1 - k2) * rN, gv = (g1 - g2) * rN;
        size_t o = (size_t)i + (size_t)j * N;
        K[o] = kv;
        G[o] = gv;
        LU[o] = kv;  // the LU buffer holds A - I/2 (lu.cu keeps the pivot's 1/2 implicit)
    }
}

// ------------------------------------------------------------------------------------------------ S1: double-double assembly
// Same formulas in dd.  sinh/cosh(eta_i - eta_j): direct series within the circular band |i-j| <= DD_BAND of the diagonal,
// addition formulas on the per-node sinh/cosh tables outside (dd has the margin: DESIGN.md section 5).
constexpr int DD_BAND = 16;
constexpr int ASMDD_TI = 128;
constexpr int ASMDD_TJ = 16;

struct NodeDD {  // per-node quantities of one collocation point
    dd eta, d1, d2, E, Dm, Sh, Ch;
    dd xE, xE1, xS, xC;  // refined mesh only (MESH): xi', xi'', sin(xi - alpha), cos(xi - alpha)
};
struct TabDD {  // functions of m = (i - j) mod N
    dd sn, cs, c0, s2;
};

// K_ij, G_ij of (2.13) in dd (already scaled by 1/N); dist = circular distance |i-j|
// rc: shared table of dd reciprocals 1 / (m (m + 1)) (fill_rc below) for the in-band series
// SLOPPY (both callers set it): sums by the 11-flop addition (error ~2^-104 relative to the LARGER operand, so a cancelling
// difference is less accurate than with the 20-flop dd_add: a cancellation by 1e3 leaves 5e-29 relative, against a bar of 1e-25 for the
// dd handles and a need of ~1e-20 in the fp64 handle's base-state pass); the argument y = eta_i - eta_j and the in-band series keep
// the accurate addition.  Entry by entry against the __float128 oracle: tests/test_gpu_parity.py, tests/test_gpu_mesh.py (1e-29 N).
__device__ __forceinline__ dd dd_add_sloppy(dd a, dd b) {
    dd s = two_sum(a.hi, b.hi);
    s.lo = SWW_ADD(s.lo, SWW_ADD(a.lo, b.lo));
    return quick_two_sum(s.hi, s.lo);
}
template <bool FINITE, bool MESH, bool SLOPPY = false>
__device__ __forceinline__ void entry_dd(const NodeDD& ni, const NodeDD& nj, const TabDD& t0, int dist, double rN, const double* rc,
                                         dd* kv, dd* gv) {
    auto add_ = [](dd a, dd b) { return SLOPPY ? dd_add_sloppy(a, b) : dd_add(a, b); };
    auto sub_ = [](dd a, dd b) { return SLOPPY ? dd_add_sloppy(a, dd_neg(b)) : dd_sub(a, b); };
    TabDD t = t0;
    if (MESH) {  // sin, cos of (alpha_i - alpha_j) + (p_i - p_j); sin^2 of half of it without cancellation
        const dd sd = sub_(dd_mul(ni.xS, nj.xC), dd_mul(ni.xC, nj.xS)), cd = add_(dd_mul(ni.xC, nj.xC), dd_mul(ni.xS, nj.xS));
        t.sn = add_(dd_mul(t0.sn, cd), dd_mul(t0.cs, sd));
        t.cs = sub_(dd_mul(t0.cs, cd), dd_mul(t0.sn, sd));
        t.s2 = t.cs.hi >= 0.0 ? dd_div(dd_sqr(t.sn), dd_mul_d(dd_add_d(t.cs, 1.0), 2.0)) : dd_half(sub_(dd{1.0, 0.0}, t.cs));
    }
    dd k1, g1;
    if (dist != 0) {
        dd sh, ch;
        const dd y = dd_sub(ni.eta, nj.eta);
        if (dist <= DD_BAND && fabs(y.hi) < 0.5) {
            dd_sinhcosh_tab(y, rc, &sh, &ch);
        } else if (dist <= DD_BAND) {
            dd_sinhcosh(y, &sh, &ch);
        } else {
            sh = sub_(dd_mul(ni.Sh, nj.Ch), dd_mul(ni.Ch, nj.Sh));
            ch = sub_(dd_mul(ni.Ch, nj.Ch), dd_mul(ni.Sh, nj.Sh));
        }
        dd p;
        if (t.cs.hi >= 0.0)
            p = dd_div_fast(add_(t.cs, ch), add_(dd_sqr(t.sn), dd_sqr(sh)));
        else
            p = dd_div_fast(dd{1.0, 0.0}, sub_(ch, t.cs));
        dd hp = dd_half(p);
        if (MESH) {
            k1 = dd_mul(hp, sub_(dd_mul(nj.d1, t.sn), dd_mul(nj.xE, sh)));
            g1 = sub_(dd_mul(hp, add_(dd_mul(ni.d1, sh), dd_mul(ni.xE, t.sn))), t.c0);
        } else {
            k1 = dd_mul(hp, sub_(dd_mul(nj.d1, t.sn), sh));
            g1 = sub_(dd_mul(hp, add_(dd_mul(ni.d1, sh), t.sn)), t.c0);
        }
    } else if (MESH) {
        dd den = dd_mul_d(add_(dd_sqr(ni.d1), dd_sqr(ni.xE)), 2.0);
        k1 = dd_neg(dd_div(sub_(dd_mul(ni.d2, ni.xE), dd_mul(ni.xE1, ni.d1)), den));
        g1 = dd_div(add_(dd_mul(ni.xE1, ni.xE), dd_mul(ni.d1, ni.d2)), den);
    } else {
        dd den = dd_mul_d(dd_add_d(dd_sqr(ni.d1), 1.0), 2.0);
        k1 = dd_neg(dd_div(ni.d2, den));
        g1 = dd_div(dd_mul(ni.d1, ni.d2), den);
    }
    dd k2{0, 0}, g2{0, 0};
    if (FINITE) {
        dd Eij = dd_mul(ni.E, nj.E);
        dd omE = add_(dd_mul(ni.E, nj.Dm), ni.Dm);
        dd den = add_(dd_sqr(omE), dd_mul_d(dd_mul(Eij, t.s2), 4.0));
        const double rb = rcp_normal(den.hi);  // both quotients share the reciprocal
        dd cr = dd_div_rb(dd_mul(Eij, t.sn), den, rb);
        dd ci = dd_neg(dd_half(dd_div_rb(dd_mul(omE, dd_add_d(Eij, 1.0)), den, rb)));
        k2 = sub_(MESH ? dd_mul(nj.xE, ci) : ci, dd_mul(nj.d1, cr));
        g2 = sub_(MESH ? dd_mul(ni.xE, cr) : cr, dd_mul(ni.d1, ci));
    }
    *kv = dd_mul_d(sub_(k1, k2), rN);
    *gv = dd_mul_d(sub_(g1, g2), rN);
}
// rc[m] (+ rc[32 + m]) = 1 / (m (m + 1)) in dd, m = 1..30; call with every thread of the CTA (ends with a barrier)
__device__ __forceinline__ void fill_rc(double* rc, int tid) {
    if (tid >= 1 && tid <= 30) {
        const dd r = dd_div(dd{1.0, 0.0}, dd{(double)(tid * (tid + 1)), 0.0});
        rc[tid] = r.hi;
        rc[32 + tid] = r.lo;
    }
    __syncthreads();
}

__device__ __forceinline__ NodeDD load_node(int N, int j, const double* eta, const double* d1, const double* d2, const double* E,
                                            const double* Dm, const double* Sh, const double* Ch, bool finite, const MeshDev& ms, bool mesh) {
    NodeDD n;
    if (mesh) {
        n.xE = dd_load(ms.xE, N, j); n.xE1 = dd_load(ms.xE1, N, j);
        n.xS = dd_load(ms.xS, N, j); n.xC = dd_load(ms.xC, N, j);
    }
    n.eta = dd_load(eta, N, j);
    n.d1 = dd_load(d1, N, j);
    n.d2 = dd_load(d2, N, j);
    n.Sh = dd_load(Sh, N, j);
    n.Ch = dd_load(Ch, N, j);
    n.E = finite ? dd_load(E, N, j) : dd{0, 0};
    n.Dm = finite ? dd_load(Dm, N, j) : dd{0, 0};
    return n;
}

template <bool FINITE, bool MESH>
__global__ void __launch_bounds__(ASMDD_TI) k_assemble_dd(int N, const double* __restrict__ eta, const double* __restrict__ d1,
                                                          const double* __restrict__ d2, const double* __restrict__ E,
                                                          const double* __restrict__ Dm, const double* __restrict__ Sh,
                                                          const double* __restrict__ Ch, const double* __restrict__ cs,
                                                          const double* __restrict__ sn, const double* __restrict__ c0,
                                                          const double* __restrict__ s2, MeshDev ms, double* __restrict__ K,
                                                          double* __restrict__ G, double* __restrict__ LU) {
    const int tid = threadIdx.x, mask = N - 1;
    const int i0 = blockIdx.x * ASMDD_TI, j0 = blockIdx.y * ASMDD_TJ;
    const int i = i0 + tid;
    __shared__ double rc[64];
    fill_rc(rc, tid);
    if (i >= N) return;
    const size_t NN = (size_t)N * N;
    const NodeDD ni = load_node(N, i, eta, d1, d2, E, Dm, Sh, Ch, FINITE, ms, MESH);
    const double rN = 1.0 / (double)N;  // exact power of two
    const int jmax = min(ASMDD_TJ, N - j0);
    for (int jj = 0; jj < jmax; jj++) {
        const int j = j0 + jj, m = (i - j) & mask;
        const NodeDD nj = load_node(N, j, eta, d1, d2, E, Dm, Sh, Ch, FINITE, ms, MESH);
        TabDD t{dd_load(sn, N, m), dd_load(cs, N, m), dd_load(c0, N, m), dd_load(s2, N, m)};
        dd kv, gv;
        entry_dd<FINITE, MESH, true>(ni, nj, t, min(m, N - m), rN, rc, &kv, &gv);
        size_t o = (size_t)i + (size_t)j * N;
        dd_store(K, NN, o, kv);
        dd_store(G, NN, o, gv);
        LU[o] = kv.hi;  // the LU buffer holds A - I/2 rounded to fp64
    }
}

// ------------------------------------------------------------------------------------------------ fused dd pass of the base state
// For the fp64 handle: the residual of (2.7) and the product with G of (2.8) for ONE vector pair (mu, gam), with the kernel
// entries evaluated in dd on the fly (nothing stored):  pK_i = sum_j K_ij mu_j ,  pG_i = sum_j G_ij gam_j  over the j-chunk of
// this CTA; partial sums go to part[chunk][4][N] (pK.hi, pK.lo, pG.hi, pG.lo) and are summed by k_base_reduce.
// Why dd: the base-state velocities u, v are multiplied into every linearized right-hand side and differentiated twice more,
// so their rounding noise is amplified by ~N^2/3.
constexpr int BP_TI = 128;
template <bool FINITE, bool MESH>
__global__ void __launch_bounds__(BP_TI) k_base_pass_dd(int N, int jchunk, const double* __restrict__ eta, const double* __restrict__ d1,
                                                        const double* __restrict__ d2, const double* __restrict__ E,
                                                        const double* __restrict__ Dm, const double* __restrict__ Sh,
                                                        const double* __restrict__ Ch, const double* __restrict__ cs,
                                                        const double* __restrict__ sn, const double* __restrict__ c0,
                                                        const double* __restrict__ s2, MeshDev ms, const double* __restrict__ mu,
                                                        const double* __restrict__ gam, double* __restrict__ part) {
    const int tid = threadIdx.x, mask = N - 1;
    const int i = blockIdx.x * BP_TI + tid, j0 = blockIdx.y * jchunk;
    __shared__ double rc[64];
    fill_rc(rc, tid);
    if (i >= N) return;
    const NodeDD ni = load_node(N, i, eta, d1, d2, E, Dm, Sh, Ch, FINITE, ms, MESH);
    const double rN = 1.0 / (double)N;
    dd aK{0, 0}, aG{0, 0};
    for (int jj = 0; jj < jchunk; jj++) {
        const int j = j0 + jj, m = (i - j) & mask;  // j is uniform over the CTA: node loads broadcast
        const NodeDD nj = load_node(N, j, eta, d1, d2, E, Dm, Sh, Ch, FINITE, ms, MESH);
        TabDD t{dd_load(sn, N, m), dd_load(cs, N, m), dd_load(c0, N, m), dd_load(s2, N, m)};
        dd kv, gv;
        entry_dd<FINITE, MESH, true>(ni, nj, t, min(m, N - m), rN, rc, &kv, &gv);
        aK = dd_fma(kv, dd_load(mu, N, j), aK);
        aG = dd_fma(gv, dd_load(gam, N, j), aG);
    }
    double* p = part + (size_t)blockIdx.y * 4 * N;
    p[i] = aK.hi;
    p[N + i] = aK.lo;
    p[2 * N + i] = aG.hi;
    p[3 * N + i] = aG.lo;
}
// ------------------------------------------------------------------------------------------------ the same pass, entries in pairs
// K_ij, G_ij and K_ji, G_ji share everything that costs: sinh/cosh(eta_i - eta_j) (odd / even under the swap), the quotient
// p = (cos x + cosh y) / (sin^2 x + sinh^2 y) (even), the image term's denominator and its two quotients c_r (odd), c_i (even).
// entry_pair_dd evaluates both entries of an off-diagonal pair for ~0.7 of the work of two entry_dd calls (11-flop additions as in
// the SLOPPY instances above).  t0: the tables of m = (i - j) mod N; dist >= 1.
template <bool FINITE, bool MESH>
__device__ __forceinline__ void entry_pair_dd(const NodeDD& ni, const NodeDD& nj, const TabDD& t0, int dist, double rN, const double* rc,
                                              dd* kij, dd* gij, dd* kji, dd* gji) {
    auto add_ = [](dd a, dd b) { return dd_add_sloppy(a, b); };
    auto sub_ = [](dd a, dd b) { return dd_add_sloppy(a, dd_neg(b)); };
    TabDD t = t0;
    if (MESH) {
        const dd sd = sub_(dd_mul(ni.xS, nj.xC), dd_mul(ni.xC, nj.xS)), cd = add_(dd_mul(ni.xC, nj.xC), dd_mul(ni.xS, nj.xS));
        t.sn = add_(dd_mul(t0.sn, cd), dd_mul(t0.cs, sd));
        t.cs = sub_(dd_mul(t0.cs, cd), dd_mul(t0.sn, sd));
        t.s2 = t.cs.hi >= 0.0 ? dd_div(dd_sqr(t.sn), dd_mul_d(dd_add_d(t.cs, 1.0), 2.0)) : dd_half(sub_(dd{1.0, 0.0}, t.cs));
    }
    dd sh, ch;
    const dd y = dd_sub(ni.eta, nj.eta);
    if (dist <= DD_BAND && fabs(y.hi) < 0.5) {
        dd_sinhcosh_tab(y, rc, &sh, &ch);
    } else if (dist <= DD_BAND) {
        dd_sinhcosh(y, &sh, &ch);
    } else {
        sh = sub_(dd_mul(ni.Sh, nj.Ch), dd_mul(ni.Ch, nj.Sh));
        ch = sub_(dd_mul(ni.Ch, nj.Ch), dd_mul(ni.Sh, nj.Sh));
    }
    dd p;
    if (t.cs.hi >= 0.0)
        p = dd_div_fast(add_(t.cs, ch), add_(dd_sqr(t.sn), dd_sqr(sh)));
    else
        p = dd_div_fast(dd{1.0, 0.0}, sub_(ch, t.cs));
    const dd hp = dd_half(p);
    // (i, j): k1 = hp (d1_j sn - xE_j sh), g1 = hp (d1_i sh + xE_i sn) - c0 ;  (j, i): sn, sh, c0 change sign, i and j change roles
    dd k1, g1, k1t, g1t;
    if (MESH) {
        k1 = dd_mul(hp, sub_(dd_mul(nj.d1, t.sn), dd_mul(nj.xE, sh)));
        g1 = sub_(dd_mul(hp, add_(dd_mul(ni.d1, sh), dd_mul(ni.xE, t.sn))), t.c0);
        k1t = dd_mul(hp, sub_(dd_mul(ni.xE, sh), dd_mul(ni.d1, t.sn)));
        g1t = sub_(t.c0, dd_mul(hp, add_(dd_mul(nj.d1, sh), dd_mul(nj.xE, t.sn))));
    } else {
        k1 = dd_mul(hp, sub_(dd_mul(nj.d1, t.sn), sh));
        g1 = sub_(dd_mul(hp, add_(dd_mul(ni.d1, sh), t.sn)), t.c0);
        k1t = dd_mul(hp, sub_(sh, dd_mul(ni.d1, t.sn)));
        g1t = sub_(t.c0, dd_mul(hp, add_(dd_mul(nj.d1, sh), t.sn)));
    }
    dd k2{0, 0}, g2{0, 0}, k2t{0, 0}, g2t{0, 0};
    if (FINITE) {
        const dd Eij = dd_mul(ni.E, nj.E);
        const dd omE = add_(dd_mul(ni.E, nj.Dm), ni.Dm);
        const dd den = add_(dd_sqr(omE), dd_mul_d(dd_mul(Eij, t.s2), 4.0));
        const double rb = rcp_normal(den.hi);
        const dd cr = dd_div_rb(dd_mul(Eij, t.sn), den, rb);
        const dd ci = dd_neg(dd_half(dd_div_rb(dd_mul(omE, dd_add_d(Eij, 1.0)), den, rb)));
        // (i, j): k2 = xE_j ci - d1_j cr, g2 = xE_i cr - d1_i ci ;  (j, i): cr changes sign
        k2 = sub_(MESH ? dd_mul(nj.xE, ci) : ci, dd_mul(nj.d1, cr));
        g2 = sub_(MESH ? dd_mul(ni.xE, cr) : cr, dd_mul(ni.d1, ci));
        k2t = add_(MESH ? dd_mul(ni.xE, ci) : ci, dd_mul(ni.d1, cr));
        g2t = dd_neg(add_(MESH ? dd_mul(nj.xE, cr) : cr, dd_mul(nj.d1, ci)));
    }
    *kij = dd_mul_d(sub_(k1, k2), rN);
    *gij = dd_mul_d(sub_(g1, g2), rN);
    *kji = dd_mul_d(sub_(k1t, k2t), rN);
    *gji = dd_mul_d(sub_(g1t, g2t), rN);
}

// BPS_NWP warps per pair of 32 x 32 tiles (Ib <= Jb) of the matrix (warp q takes the steps s = 8 q .. 8 q + 7; their sums meet in shared
// memory -- the 8320 quarter-size units at N = 2048 fill the resident warps of the chip more evenly than 2080 full ones): lane l owns row i = 32 Ib + l and meets the columns j = 32 Jb + ((l + s) mod 32) (each step the 32 lanes hold
// 32 different columns).  The row sums stay with the lane; the sums for the rows j (from
// the transposed entries K_ji, G_ji) travel with their column from lane to lane by shuffles and end where they started.  Output in the
// layout of k_base_pass_dd with column chunks of 32: part[Jb][.][rows of Ib] and part[Ib][.][rows of Jb], every slot written once.
// Diagonal tiles (Ib == Jb) take the plain entries (they hold i == j).  N a multiple of 32; nT = N / 32.
constexpr int BPS_WARPS = 4;   // warps per CTA
constexpr int BPS_NWP = 4;     // warps per tile pair: each takes 32 / BPS_NWP of the 32 steps
template <bool FINITE, bool MESH>
__global__ void __launch_bounds__(32 * BPS_WARPS) k_base_pass_sym(int N, int nT, const double* __restrict__ eta, const double* __restrict__ d1,
                                                                  const double* __restrict__ d2, const double* __restrict__ E,
                                                                  const double* __restrict__ Dm, const double* __restrict__ Sh,
                                                                  const double* __restrict__ Ch, const double* __restrict__ cs,
                                                                  const double* __restrict__ sn, const double* __restrict__ c0,
                                                                  const double* __restrict__ s2, MeshDev ms, const double* __restrict__ mu,
                                                                  const double* __restrict__ gam, double* __restrict__ part) {
    constexpr int NF = MESH ? 26 : 18;  // doubles per staged node: 7 dd fields, mu, gam (+ 4 dd mesh fields)
    constexpr int NP = BPS_WARPS / BPS_NWP, NS = 32 / BPS_NWP;  // tile pairs per CTA, steps per warp
    __shared__ double rc[64];
    __shared__ double sJ[NP][NF][32];
    __shared__ double sX[NP][BPS_NWP][8][32];  // the other warps' sums on their way to the first: rows (4), columns (4, by column)
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, mask = N - 1, pr_ = warp / BPS_NWP, half = warp % BPS_NWP;
    fill_rc(rc, tid);
    int u = blockIdx.x * NP + pr_, Ib = 0;
    const int nunits = nT * (nT + 1) / 2;
    const bool live = u < nunits;       // (a CTA's warps all reach the barriers below)
    if (!live) u = 0;
    while (u >= nT - Ib) {
        u -= nT - Ib;
        Ib++;
    }
    const int Jb = Ib + u, i = 32 * Ib + lane;
    const NodeDD ni = load_node(N, i, eta, d1, d2, E, Dm, Sh, Ch, FINITE, ms, MESH);
    const dd mu_i = dd_load(mu, N, i), gam_i = dd_load(gam, N, i);
    if (half == 0) {   // stage the nodes of the column tile
        const int j = 32 * Jb + lane;
        const NodeDD n = load_node(N, j, eta, d1, d2, E, Dm, Sh, Ch, FINITE, ms, MESH);
        double(*f)[32] = sJ[pr_];
        f[0][lane] = n.eta.hi; f[1][lane] = n.eta.lo; f[2][lane] = n.d1.hi; f[3][lane] = n.d1.lo; f[4][lane] = n.d2.hi; f[5][lane] = n.d2.lo;
        f[6][lane] = n.E.hi; f[7][lane] = n.E.lo; f[8][lane] = n.Dm.hi; f[9][lane] = n.Dm.lo; f[10][lane] = n.Sh.hi; f[11][lane] = n.Sh.lo;
        f[12][lane] = n.Ch.hi; f[13][lane] = n.Ch.lo;
        const dd m_ = dd_load(mu, N, j), g_ = dd_load(gam, N, j);
        f[14][lane] = m_.hi; f[15][lane] = m_.lo; f[16][lane] = g_.hi; f[17][lane] = g_.lo;
        if (MESH) {
            f[18][lane] = n.xE.hi; f[19][lane] = n.xE.lo; f[20][lane] = n.xE1.hi; f[21][lane] = n.xE1.lo;
            f[22][lane] = n.xS.hi; f[23][lane] = n.xS.lo; f[24][lane] = n.xC.hi; f[25][lane] = n.xC.lo;
        }
    }
    __syncthreads();
    const double rN = 1.0 / (double)N;
    const bool diag = Ib == Jb;
    dd aK{0, 0}, aG{0, 0}, tK{0, 0}, tG{0, 0};
    for (int s = NS * half; s < NS * half + NS; s++) {
        const int jl = (lane + s) & 31, j = 32 * Jb + jl, m = (i - j) & mask;
        const double(*f)[32] = sJ[pr_];
        NodeDD nj;
        nj.eta = dd{f[0][jl], f[1][jl]}; nj.d1 = dd{f[2][jl], f[3][jl]}; nj.d2 = dd{f[4][jl], f[5][jl]};
        nj.E = dd{f[6][jl], f[7][jl]}; nj.Dm = dd{f[8][jl], f[9][jl]}; nj.Sh = dd{f[10][jl], f[11][jl]}; nj.Ch = dd{f[12][jl], f[13][jl]};
        if (MESH) {
            nj.xE = dd{f[18][jl], f[19][jl]}; nj.xE1 = dd{f[20][jl], f[21][jl]};
            nj.xS = dd{f[22][jl], f[23][jl]}; nj.xC = dd{f[24][jl], f[25][jl]};
        }
        const dd mu_j{f[14][jl], f[15][jl]}, gam_j{f[16][jl], f[17][jl]};
        const TabDD t{dd_load(sn, N, m), dd_load(cs, N, m), dd_load(c0, N, m), dd_load(s2, N, m)};
        if (diag) {
            dd kv, gv;
            entry_dd<FINITE, MESH, true>(ni, nj, t, min(m, N - m), rN, rc, &kv, &gv);
            aK = dd_fma(kv, mu_j, aK);
            aG = dd_fma(gv, gam_j, aG);
        } else {
            dd kij, gij, kji, gji;
            entry_pair_dd<FINITE, MESH>(ni, nj, t, min(m, N - m), rN, rc, &kij, &gij, &kji, &gji);
            aK = dd_fma(kij, mu_j, aK);
            aG = dd_fma(gij, gam_j, aG);
            tK = dd_fma(kji, mu_i, tK);
            tG = dd_fma(gji, gam_i, tG);
            // the sums of column j move on with it: the lane below meets this column next
            const int src = (lane + 1) & 31;
            tK = dd{__shfl_sync(0xffffffffu, tK.hi, src), __shfl_sync(0xffffffffu, tK.lo, src)};
            tG = dd{__shfl_sync(0xffffffffu, tG.hi, src), __shfl_sync(0xffffffffu, tG.lo, src)};
        }
    }
    // after its NS moves a lane holds the sums of column (lane + NS (half + 1)) mod 32
    const int c = (lane + NS * (half + 1)) & 31;
    if (half != 0) {
        double(*x)[32] = sX[pr_][half];
        x[0][lane] = aK.hi; x[1][lane] = aK.lo; x[2][lane] = aG.hi; x[3][lane] = aG.lo;
        x[4][c] = tK.hi; x[5][c] = tK.lo; x[6][c] = tG.hi; x[7][c] = tG.lo;
    }
    __syncthreads();
    if (half != 0 || !live) return;
    for (int q = 1; q < BPS_NWP; q++) {
        const double(*x)[32] = sX[pr_][q];
        aK = dd_add(aK, dd{x[0][lane], x[1][lane]});
        aG = dd_add(aG, dd{x[2][lane], x[3][lane]});
        if (!diag) {
            tK = dd_add(tK, dd{x[4][c], x[5][c]});
            tG = dd_add(tG, dd{x[6][c], x[7][c]});
        }
    }
    double* pr = part + (size_t)Jb * 4 * N;   // rows of Ib, columns of chunk Jb
    pr[i] = aK.hi; pr[N + i] = aK.lo; pr[2 * N + i] = aG.hi; pr[3 * N + i] = aG.lo;
    if (!diag) {                              // rows of Jb, columns of chunk Ib
        const int j = 32 * Jb + c;
        double* pc = part + (size_t)Ib * 4 * N;
        pc[j] = tK.hi; pc[N + j] = tK.lo; pc[2 * N + j] = tG.hi; pc[3 * N + j] = tG.lo;
    }
}

// res = b - mu/2 - sum pK  (2.7) ;  w = sum pG ;  res_f64 = RN(res).  512 threads = 32 nodes x 16 groups of chunks (the loads of a
// node's partial sums are the whole cost: sixteen groups keep sixteen of them in flight and shorten the dd chains).
constexpr int BR_G = 16;
__global__ void __launch_bounds__(32 * BR_G) k_base_reduce(int N, int nchunk, const double* __restrict__ part, const double* __restrict__ b,
                                                           const double* __restrict__ mu, double* __restrict__ res, double* __restrict__ res_f64,
                                                           double* __restrict__ w) {
    __shared__ double sh[BR_G][4][32];
    const int l = threadIdx.x & 31, g = threadIdx.x >> 5;
    const int i = blockIdx.x * 32 + l;
    dd sK{0, 0}, sG{0, 0};
    if (i < N) {
        for (int c = g; c < nchunk; c += BR_G) {
            const double* p = part + (size_t)c * 4 * N;
            sK = dd_add(sK, dd{p[i], p[N + i]});
            sG = dd_add(sG, dd{p[2 * N + i], p[3 * N + i]});
        }
    }
    sh[g][0][l] = sK.hi; sh[g][1][l] = sK.lo; sh[g][2][l] = sG.hi; sh[g][3][l] = sG.lo;
    __syncthreads();
    if (g != 0 || i >= N) return;
    for (int q = 1; q < BR_G; q++) {
        sK = dd_add(sK, dd{sh[q][0][l], sh[q][1][l]});
        sG = dd_add(sG, dd{sh[q][2][l], sh[q][3][l]});
    }
    dd r = dd_sub(dd_sub(dd_load(b, N, i), dd_half(dd_load(mu, N, i))), sK);
    dd_store(res, N, i, r);
    res_f64[i] = r.hi;
    dd_store(w, N, i, sG);
}

int base_pass_dd(sww_dtn_s* d, const double* b, const double* mu, const double* gam, double* res, double* res_f64, double* w) {
    const int N = d->N;
    const Tables* t = d->tab;
    int nchunk = d->bp_chunks;
    const int jchunk = N / nchunk;
    dim3 grid((N + BP_TI - 1) / BP_TI, nchunk);
    SWW_BEGIN(KC_DDGEMM, d->stream);
    const MeshDev ms = d->mesh;
    if (N >= 2048 && N / 32 <= d->bp_chunks) {  // enough tile pairs to fill the chip: the entries in pairs (k_base_pass_sym)
        const int nT = N / 32, nunits = nT * (nT + 1) / 2;
        const dim3 gs((nunits + BPS_WARPS / BPS_NWP - 1) / (BPS_WARPS / BPS_NWP));
#define SWW_BPS_LAUNCH(FIN, MSH) \
    k_base_pass_sym<FIN, MSH><<<gs, 32 * BPS_WARPS, 0, d->stream>>>(N, nT, d->eta, d->d1, d->d2, d->E, d->Dm, d->Sh, d->Ch, t->cs, t->sn, t->c0, t->s2, ms, mu, gam, d->bp_part)
        if (d->mesh_on) {
            if (d->finite) SWW_BPS_LAUNCH(true, true); else SWW_BPS_LAUNCH(false, true);
        } else {
            if (d->finite) SWW_BPS_LAUNCH(true, false); else SWW_BPS_LAUNCH(false, false);
        }
#undef SWW_BPS_LAUNCH
        nchunk = nT;
        SWW_LAUNCHED();
        SWW_BEGIN(KC_OTHER, d->stream);
        k_base_reduce<<<(N + 31) / 32, 32 * BR_G, 0, d->stream>>>(N, nchunk, d->bp_part, b, mu, res, res_f64, w);
        SWW_LAUNCHED();
        SWW_CUDA(cudaGetLastError());
        return SWW_OK;
    }
#define SWW_BP_LAUNCH(FIN, MSH) \
    k_base_pass_dd<FIN, MSH><<<grid, BP_TI, 0, d->stream>>>(N, jchunk, d->eta, d->d1, d->d2, d->E, d->Dm, d->Sh, d->Ch, t->cs, t->sn, t->c0, t->s2, ms, mu, gam, d->bp_part)
    if (d->mesh_on) {
        if (d->finite) SWW_BP_LAUNCH(true, true); else SWW_BP_LAUNCH(false, true);
    } else {
        if (d->finite) SWW_BP_LAUNCH(true, false); else SWW_BP_LAUNCH(false, false);
    }
#undef SWW_BP_LAUNCH
    SWW_LAUNCHED();
    SWW_BEGIN(KC_OTHER, d->stream);
    k_base_reduce<<<(N + 31) / 32, 32 * BR_G, 0, d->stream>>>(N, nchunk, d->bp_part, b, mu, res, res_f64, w);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

static int run_node_prep(sww_dtn_s* d) {
    const int N = d->N;
    cudaStream_t st = d->stream;
    SWW_BEGIN(KC_OTHER, st);
    k_node_prep<<<(N + 1) / 2, 256, 0, st>>>(N, d->h, d->finite ? 1 : 0, d->tab->dc, d->tab->dc2, d->eta, d->d1, d->d2, d->E, d->Dm, d->Sh, d->Ch,
                                              d->status);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

int run_setup_f64(sww_dtn_s* d) {
    SWW_TRY(run_node_prep(d));
    const int N = d->N;
    const Tables* t = d->tab;
    // sources per CTA: 32, or 4 at small N (N = 256 would otherwise run on 16 CTAs)
    const int tj = (N <= 512) ? 4 : ASM_TJ;
    dim3 grid((N + ASM_TI - 1) / ASM_TI, (N + tj - 1) / tj);
    SWW_BEGIN(KC_ASM, d->stream);
    const MeshDev ms = d->mesh;
#define SWW_ASM_LAUNCH(FIN, TJV, MSH) \
    k_assemble_f64<FIN, TJV, MSH><<<grid, ASM_TI, 0, d->stream>>>(N, d->eta, d->d1, d->d2, d->E, d->Dm, t->cs, t->sn, t->c0, t->s2, ms, d->K, d->G, d->LU)
    if (d->mesh_on) {
        if (d->finite) {
            if (tj == 4) SWW_ASM_LAUNCH(true, 4, true); else SWW_ASM_LAUNCH(true, ASM_TJ, true);
        } else {
            if (tj == 4) SWW_ASM_LAUNCH(false, 4, true); else SWW_ASM_LAUNCH(false, ASM_TJ, true);
        }
    } else if (d->finite) {
        if (tj == 4) SWW_ASM_LAUNCH(true, 4, false); else SWW_ASM_LAUNCH(true, ASM_TJ, false);
    } else {
        if (tj == 4) SWW_ASM_LAUNCH(false, 4, false); else SWW_ASM_LAUNCH(false, ASM_TJ, false);
    }
#undef SWW_ASM_LAUNCH
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

int run_setup_dd(sww_dtn_s* d) {
    SWW_TRY(run_node_prep(d));
    const int N = d->N;
    const Tables* t = d->tab;
    dim3 grid((N + ASMDD_TI - 1) / ASMDD_TI, (N + ASMDD_TJ - 1) / ASMDD_TJ);
    SWW_BEGIN(KC_ASM, d->stream);
    const MeshDev ms = d->mesh;
#define SWW_ASMDD_LAUNCH(FIN, MSH) \
    k_assemble_dd<FIN, MSH><<<grid, ASMDD_TI, 0, d->stream>>>(N, d->eta, d->d1, d->d2, d->E, d->Dm, d->Sh, d->Ch, t->cs, t->sn, t->c0, t->s2, ms, d->K, d->G, d->LU)
    if (d->mesh_on) {
        if (d->finite) SWW_ASMDD_LAUNCH(true, true); else SWW_ASMDD_LAUNCH(false, true);
    } else {
        if (d->finite) SWW_ASMDD_LAUNCH(true, false); else SWW_ASMDD_LAUNCH(false, false);
    }
#undef SWW_ASMDD_LAUNCH
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

}  // namespace sww
