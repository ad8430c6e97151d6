// lm.cu -- Levenberg-Marquardt with delayed Jacobian updates (Appendix C, 751-818) around the device shooting map.
// HOST code: the small dense algebra of the outer solver (thin SVD of the N x m Jacobian via Householder QR + one-sided Jacobi on
// the m x m factor, the O(m) Newton iteration (C.5) for the Lagrange multiplier, the trust-region bookkeeping of rules 1-4).
// Every residual and Jacobian comes from a callback; sww_lm_shoot plugs in sww_shoot (device: time stepping with the batched
// linearized DtN), which is where the time goes.  Product code; shares nothing with oracle/.
#include "common.cuh"
#include <algorithm>
#include <cmath>
#include <cstring>
#include <vector>

namespace sww {

// ---- thin SVD  J = U S V^T  of an M x m matrix (column-major, M >= m), in the form the iteration needs:
// on return  Rt = U^T r (m),  sig (m),  V (m x m column-major).  J and r are overwritten.
// Householder QR of [J | r] (so U^T r = Ur^T (Q^T r) without forming Q), then one-sided Jacobi (Hestenes) on R.
static void svd_thin(int M, int m, std::vector<double>& J, std::vector<double>& r, std::vector<double>& sig, std::vector<double>& V,
                     std::vector<double>& Rt) {
    std::vector<double> R((size_t)m * m, 0.0);
    for (int k = 0; k < m; k++) {
        double* a = &J[(size_t)k * M];
        long double nrm2 = 0.0L;
        for (int i = k; i < M; i++) nrm2 += (long double)a[i] * a[i];
        const double nrm = (double)sqrtl(nrm2);
        if (nrm == 0.0) continue;  // zero column: R_kk = 0
        const double alpha = a[k] > 0 ? -nrm : nrm;
        std::vector<double> v(a + k, a + M);
        v[0] -= alpha;
        long double vv = 0.0L;
        for (double x : v) vv += (long double)x * x;
        if (vv == 0.0L) continue;
        auto reflect = [&](double* col) {  // col[k..M) -= 2 v (v . col) / (v . v)
            long double dot = 0.0L;
            for (int i = k; i < M; i++) dot += (long double)v[i - k] * col[i];
            const double s = (double)(2.0L * dot / vv);
            for (int i = k; i < M; i++) col[i] -= s * v[i - k];
        };
        for (int j = k; j < m; j++) reflect(&J[(size_t)j * M]);
        reflect(r.data());
    }
    for (int j = 0; j < m; j++)
        for (int i = 0; i <= j; i++) R[(size_t)j * m + i] = J[(size_t)j * M + i];
    // one-sided Jacobi on R: rotate column pairs until orthogonal; W = R V has orthogonal columns, sig = column norms, Ur = W / sig
    V.assign((size_t)m * m, 0.0);
    for (int i = 0; i < m; i++) V[(size_t)i * m + i] = 1.0;
    for (int sweep = 0; sweep < 60; sweep++) {
        double off = 0.0;
        for (int p = 0; p < m - 1; p++)
            for (int q = p + 1; q < m; q++) {
                double* a = &R[(size_t)p * m];
                double* b = &R[(size_t)q * m];
                long double app = 0, aqq = 0, apq = 0;
                for (int i = 0; i < m; i++) {
                    app += (long double)a[i] * a[i];
                    aqq += (long double)b[i] * b[i];
                    apq += (long double)a[i] * b[i];
                }
                if (apq == 0.0L) continue;
                const double rel = (double)(fabsl(apq) / sqrtl(app * aqq + 1e-600L));
                off = std::max(off, rel);
                if (rel < 1e-17) continue;
                const long double zeta = (aqq - app) / (2.0L * apq);
                const long double t = (zeta >= 0 ? 1.0L : -1.0L) / (fabsl(zeta) + sqrtl(1.0L + zeta * zeta));
                const double cs = (double)(1.0L / sqrtl(1.0L + t * t)), sn = (double)(cs * t);
                for (int i = 0; i < m; i++) {
                    const double x = a[i], y = b[i];
                    a[i] = cs * x - sn * y;
                    b[i] = sn * x + cs * y;
                }
                double* vp = &V[(size_t)p * m];
                double* vq = &V[(size_t)q * m];
                for (int i = 0; i < m; i++) {
                    const double x = vp[i], y = vq[i];
                    vp[i] = cs * x - sn * y;
                    vq[i] = sn * x + cs * y;
                }
            }
        if (off < 1e-16) break;
    }
    sig.assign(m, 0.0);
    Rt.assign(m, 0.0);
    for (int k = 0; k < m; k++) {
        const double* w = &R[(size_t)k * m];
        long double s2 = 0, d = 0;
        for (int i = 0; i < m; i++) {
            s2 += (long double)w[i] * w[i];
            d += (long double)w[i] * r[i];   // r now holds Q^T r; its first m entries are what U^T needs
        }
        sig[k] = (double)sqrtl(s2);
        Rt[k] = sig[k] > 0 ? (double)(d / sqrtl(s2)) : 0.0;
    }
}

// (C.3)-(C.5): p~ = argmin || [S; sqrt(lambda) I] p~ + [r~; 0] ||  =>  p~_k = -sig_k r~_k / (sig_k^2 + lambda); Newton on tau(lambda)
static void tr_step(int m, const std::vector<double>& sig, const std::vector<double>& rt, double Delta, double tol, std::vector<double>& pt,
                    double& lambda) {
    lambda = 0.0;
    pt.assign(m, 0.0);
    double smax = 0.0;
    for (double s : sig) smax = std::max(smax, s);
    const double floor2 = (smax * 1e-300) * (smax * 1e-300);
    auto solve = [&](double lam) {
        long double n2 = 0;
        for (int k = 0; k < m; k++) {
            const double den = sig[k] * sig[k] + lam;
            pt[k] = den > floor2 ? -sig[k] * rt[k] / den : 0.0;
            n2 += (long double)pt[k] * pt[k];
        }
        return (double)sqrtl(n2);
    };
    double np = solve(0.0);
    for (int l = 0; l < 200 && (np - Delta) / Delta > tol; l++) {
        long double num = 0, den = 0;
        for (int k = 0; k < m; k++) {
            if (pt[k] == 0.0) continue;   // directions with sigma = 0 carry no step
            num += (long double)pt[k] * pt[k];
            den += (long double)pt[k] * pt[k] / (sig[k] * sig[k] + lambda);   // p~^T (S^T S + lambda I)^-1 p~: Newton on tau (R14)
        }
        if (!(den > 0) || !std::isfinite((double)den)) break;
        lambda += (double)(num / den) * ((np - Delta) / Delta);
        np = solve(lambda);
    }
}

}  // namespace sww

using namespace sww;

extern "C" {

// fun(ctx, c, want_J, r, J): residual r (M) and, when want_J, the Jacobian (M x ntot column-major, all unknowns) at c; 0 on success
int sww_lm_minimize(sww_lm_fun fun, void* ctx, int M, int ntot, double* c, const int* fixed, const sww_lm_options* opt, sww_lm_report* rep) {
    if (!fun || !c || M < 1 || ntot < 1 || !opt) return SWW_EINVAL;
    std::vector<int> free_idx;
    for (int k = 0; k < ntot; k++)
        if (!fixed || !fixed[k]) free_idx.push_back(k);
    const int m = (int)free_idx.size();
    if (m < 1 || m > M) return SWW_EINVAL;
    const double f_tol = opt->f_tol, g_tol = opt->g_tol, df_tol = opt->df_tol;
    const int max_stepsJ = opt->max_stepsJ > 0 ? opt->max_stepsJ : 10, max_iter = opt->max_iter > 0 ? opt->max_iter : 100;
    const double rho0 = 0.25, rho1 = 0.85, a0 = 0.375, a1 = 1.875, a2 = 0.2;   // rule 2, (C.6)
    std::vector<double> r(M), rn(M), Jfull((size_t)M * ntot), J, sig, V, rt, pt, p(m), cn(ntot), rwork;
    auto half_norm2 = [&](const std::vector<double>& v) {
        long double s = 0;
        for (double x : v) s += (long double)x * x;
        return (double)(0.5L * s);
    };
    int nres = 0, njac = 0, iters = 0, rc = 0;
    double Delta = opt->delta0 > 0 ? opt->delta0 : 1.0;
    bool roundoff = false, haveJ = false, first_rej_set = false;
    double delta_first_rejected = 0.0, delta_trigger = 0.0;
    int stepsJ = 0;
    double f = 0.0, gnorm = 0.0;
    auto eval = [&](const double* cc, bool wantJ, std::vector<double>& rout) {
        const int e = fun(ctx, cc, wantJ ? 1 : 0, rout.data(), wantJ ? Jfull.data() : nullptr);
        if (wantJ) njac++;
        else nres++;
        return e;
    };
    auto factor = [&]() {  // J (free columns) -> SVD; rt = U^T r
        J.resize((size_t)M * m);
        for (int q = 0; q < m; q++) memcpy(&J[(size_t)q * M], &Jfull[(size_t)free_idx[q] * M], sizeof(double) * M);
        // g = J^T r before J is overwritten
        long double g2 = 0;
        for (int q = 0; q < m; q++) {
            long double d = 0;
            for (int i = 0; i < M; i++) d += (long double)J[(size_t)q * M + i] * r[i];
            g2 += d * d;
        }
        gnorm = (double)sqrtl(g2);
        rwork = r;
        svd_thin(M, m, J, rwork, sig, V, rt);
        haveJ = true;
        stepsJ = 0;
        first_rej_set = false;
    };
    // r~ for the current residual with the stored factorisation: U^T r needs U; U = J V S^-1 is not kept, so when J is re-used the
    // projection is rebuilt from the kept copy of the free columns: r~ = S^-1 V^T (J^T r)
    std::vector<double> Jkeep;
    auto project = [&](const std::vector<double>& rv) {
        std::vector<double> g(m);
        for (int q = 0; q < m; q++) {
            long double d = 0;
            for (int i = 0; i < M; i++) d += (long double)Jkeep[(size_t)q * M + i] * rv[i];
            g[q] = (double)d;
        }
        for (int k = 0; k < m; k++) {
            long double d = 0;
            for (int q = 0; q < m; q++) d += (long double)V[(size_t)k * m + q] * g[q];
            rt[k] = sig[k] > 0 ? (double)(d / sig[k]) : 0.0;
        }
    };
    rc = eval(c, true, r);
    if (rc) return rc;
    f = half_norm2(r);
    Jkeep.resize((size_t)M * m);
    for (int q = 0; q < m; q++) memcpy(&Jkeep[(size_t)q * M], &Jfull[(size_t)free_idx[q] * M], sizeof(double) * M);
    factor();
    int status = 0;  // 0: iteration limit, 1: f = 0, 2: c unchanged, 3: roundoff regime ended
    for (iters = 0; iters < max_iter; iters++) {
        if (f == 0.0) { status = 1; break; }
        double lambda = 0.0;
        tr_step(m, sig, rt, Delta, opt->lambda_tol > 0 ? opt->lambda_tol : 1e-12, pt, lambda);
        long double pn2 = 0, df = 0;
        for (int k = 0; k < m; k++) {   // df = g~.p~ + p~ S^2 p~ / 2 with g~ = S r~
            pn2 += (long double)pt[k] * pt[k];
            df += (long double)sig[k] * rt[k] * pt[k] + 0.5L * (long double)sig[k] * sig[k] * pt[k] * pt[k];
        }
        const double pnorm = (double)sqrtl(pn2);
        for (int q = 0; q < m; q++) {   // p = V p~
            long double d = 0;
            for (int k = 0; k < m; k++) d += (long double)V[(size_t)k * m + q] * pt[k];
            p[q] = (double)d;
        }
        if (stepsJ == 0 && (gnorm < g_tol || fabs((double)df) / f < df_tol)) roundoff = true;   // rule 1
        if (f < f_tol || Delta < g_tol) roundoff = true;
        cn.assign(c, c + ntot);
        bool changed = false;
        for (int q = 0; q < m; q++) {
            const double v = cn[free_idx[q]] + p[q];
            changed |= v != cn[free_idx[q]];
            cn[free_idx[q]] = v;
        }
        if (!changed) { status = 2; break; }
        rc = eval(cn.data(), false, rn);
        if (rc) return rc;
        const double fn = half_norm2(rn);
        const double rho = df < 0 ? (fn - f) / (double)df : -1.0;   // rule 2: actual / predicted change (the latter negative)
        const bool accept = rho > 0;
        if (rho < rho0) {
            if (!first_rej_set) { delta_first_rejected = Delta; delta_trigger = a2 * Delta; first_rej_set = true; }
            Delta = a0 * pnorm;
        } else if (rho > rho1 && pnorm > 0.9 * Delta) {
            Delta *= a1;
        }
        if (accept) {
            memcpy(c, cn.data(), sizeof(double) * ntot);
            r = rn;
            f = fn;
            stepsJ++;
            if (rho >= rho0) first_rej_set = false;   // "the first rejected radius after (or coinciding with) an accepted step"
        }
        if (roundoff && (!accept || stepsJ >= max_stepsJ)) { status = 3; break; }
        // rule 3: when to recompute J
        bool recompute = false;
        if (!roundoff) {
            if (stepsJ >= max_stepsJ) recompute = true;
            if (stepsJ > 0 && first_rej_set && Delta < delta_trigger) recompute = true;
            if (stepsJ > 0 && accept) {
                project(r);
                long double dfn = 0;
                std::vector<double> ptn;
                double lam;
                tr_step(m, sig, rt, Delta, 1e-12, ptn, lam);
                for (int k = 0; k < m; k++) dfn += (long double)sig[k] * rt[k] * ptn[k] + 0.5L * (long double)sig[k] * sig[k] * ptn[k] * ptn[k];
                if (f > 0 && fabs((double)dfn) / f < df_tol) recompute = true;
            }
        }
        if (recompute) {
            if (first_rej_set) Delta = delta_first_rejected / a1;
            rc = eval(c, true, r);
            if (rc) return rc;
            f = half_norm2(r);
            for (int q = 0; q < m; q++) memcpy(&Jkeep[(size_t)q * M], &Jfull[(size_t)free_idx[q] * M], sizeof(double) * M);
            factor();
        } else if (accept) {
            project(r);   // rule 4: r only; the old factorisation serves the next step
        }
    }
    if (rep) {
        rep->f = f;
        rep->iterations = iters;
        rep->residual_evals = nres;
        rep->jacobian_evals = njac;
        rep->status = status;
        rep->delta = Delta;
    }
    return SWW_OK;
}

}  // extern "C"

// ---- the shooting map as the callback
struct ShootCtx {
    sww_shooter_t S;
    int N, n, nsteps, isdd;
    double *r_dev, *J_dev;
    std::vector<double> tmp;
};

static int shoot_fun(void* vctx, const double* c, int want_J, double* r, double* J) {
    ShootCtx* x = (ShootCtx*)vctx;
    const int N = x->N, n = x->n;
    int rc = want_J ? sww_shoot(x->S, c, x->nsteps, x->r_dev, x->J_dev, nullptr, nullptr) : sww_shoot_residual(x->S, c, x->nsteps, x->r_dev);
    if (rc) return rc;
    // double-double outputs are read as hi + lo rounded to fp64: the iteration's algebra is fp64 (c itself is fp64)
    const size_t nr = (size_t)N * (x->isdd ? 2 : 1), nj = (size_t)N * (n + 1) * (x->isdd ? 2 : 1);
    x->tmp.resize(std::max(nr, nj));
    if (cudaMemcpy(x->tmp.data(), x->r_dev, sizeof(double) * nr, cudaMemcpyDeviceToHost) != cudaSuccess) return SWW_ECUDA;
    for (int i = 0; i < N; i++) r[i] = x->isdd ? x->tmp[i] + x->tmp[N + i] : x->tmp[i];
    if (want_J) {
        if (cudaMemcpy(x->tmp.data(), x->J_dev, sizeof(double) * nj, cudaMemcpyDeviceToHost) != cudaSuccess) return SWW_ECUDA;
        const size_t L = (size_t)N * (n + 1);
        for (size_t i = 0; i < L; i++) J[i] = x->isdd ? x->tmp[i] + x->tmp[L + i] : x->tmp[i];
    }
    return 0;
}

extern "C" int sww_lm_shoot(sww_shooter_t S, double* c, const int* fixed, int nsteps, const sww_lm_options* opt, sww_lm_report* rep) {
    if (!S || !c || nsteps < 1 || !opt) return SWW_EINVAL;
    ShootCtx x;
    x.S = S;
    sww_shooter_dims(S, &x.N, &x.n, &x.isdd);
    x.nsteps = nsteps;
    const size_t mul = x.isdd ? 2 : 1;
    x.r_dev = x.J_dev = nullptr;
    if (cudaMalloc(&x.r_dev, sizeof(double) * mul * x.N) != cudaSuccess || cudaMalloc(&x.J_dev, sizeof(double) * mul * x.N * (x.n + 1)) != cudaSuccess) {
        cudaFree(x.r_dev);
        return SWW_ENOMEM;
    }
    const int rc = sww_lm_minimize(shoot_fun, &x, x.N, x.n + 1, c, fixed, opt, rep);
    cudaFree(x.r_dev);
    cudaFree(x.J_dev);
    return rc;
}
