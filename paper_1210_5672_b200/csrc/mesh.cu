// mesh.cu -- mesh refinement in space, PAPER.md:122-136:
//   (2.10) the change of variables x = xi(alpha), xi' = E = 1 - P[A sin^4(alpha/2)] (refine near x = pi) or 1 - P[A cos^4(alpha/2)]
//          (refine near x = 0), A = 8 (1 - rho) / (5 + 3 rho); (2.11) rho = min E / max E.  With sin^4(a/2) = 3/8 - cos(a)/2 + cos(2a)/8:
//              E = 1 + a1 cos(alpha) + a2 cos(2 alpha),  xi - alpha = a1 sin(alpha) + (a2/2) sin(2 alpha),  a1 = +-A/2, a2 = -A/8.
//   The state is stored at the points x_j = xi(alpha_j) of a uniform alpha-mesh; zeta = xi + i eta o xi in (2.13) (assembly.cu),
//   the factor 1/|xi'| of (2.8) and d/dx = (1/xi') d/dalpha elsewhere (api.cu, ddpath.cu, rk.cu).
//   Respacing between segments: f o xi_new(alpha_j) = (f o xi_old)(beta_j), beta_j = xi_old^{-1}(xi_new(alpha_j)) by
//   Newton's method; the values at beta_j come from the trigonometric interpolant of the old samples, written as one matrix
//   R (M_new x M_old, the periodic Dirichlet kernel) applied to all state columns at once by the library's fp64 GEMM (double-double
//   states: the matrix and the product in double-double).
// Product code; shares nothing with oracle/.
#include "rk.cuh"
#include "dd.cuh"
#include <cmath>

using namespace sww;

namespace sww {

// A = 8 (1 - rho) / (5 + 3 rho) in double-double (rho is an fp64 number; every operation below is exact or a dd operation)
__device__ __forceinline__ dd mesh_A(double rho) {
    const dd num = dd_mul_d(two_sum(1.0, -rho), 8.0);
    const dd den = dd_add_d(two_prod(3.0, rho), 5.0);
    return dd_div(num, den);
}

// sin and cos of a dd angle of any moderate size: reduce by multiples of pi/2, then the Taylor series of dd.cuh
__device__ inline void dd_sincos_any(dd x, dd* s, dd* c) {
    const dd hp = dd_half(dd_pi());
    const double kf = rint(x.hi / hp.hi);
    const dd r = dd_sub(x, dd_mul_d(hp, kf));
    dd ss, cc;
    dd_sincos_small(r, &ss, &cc);
    switch (((long long)kf) & 3) {
        case 0: *s = ss; *c = cc; break;
        case 1: *s = cc; *c = dd_neg(ss); break;
        case 2: *s = dd_neg(ss); *c = dd_neg(cc); break;
        default: *s = dd_neg(cc); *c = ss; break;
    }
}

// per-node tables of the handle: xE, xE1, xS, xC (dd planar 2N each), from the exact per-N tables cs, sn of cos, sin(2 pi m / N)
__global__ void k_mesh_tables(int N, double rho, int where, const double* __restrict__ cs, const double* __restrict__ sn, double* __restrict__ xE,
                              double* __restrict__ xE1, double* __restrict__ xS, double* __restrict__ xC, double* __restrict__ coef) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    const dd A = mesh_A(rho);
    const dd a1 = where == 0 ? dd_half(A) : dd_neg(dd_half(A)), a2 = dd_neg(dd_ldexp(A, -3));
    if (j == 0) {
        coef[0] = a1.hi; coef[1] = a1.lo; coef[2] = a2.hi; coef[3] = a2.lo;
    }
    const int j2 = (2 * j) & (N - 1);
    const dd c1 = dd_load(cs, N, j), s1 = dd_load(sn, N, j), c2 = dd_load(cs, N, j2), s2 = dd_load(sn, N, j2);
    dd_store(xE, N, j, dd_add(dd_add_d(dd_mul(a1, c1), 1.0), dd_mul(a2, c2)));
    dd_store(xE1, N, j, dd_neg(dd_add(dd_mul(a1, s1), dd_mul(dd_mul_d(a2, 2.0), s2))));
    const dd p = dd_add(dd_mul(a1, s1), dd_mul(dd_half(a2), s2));
    dd S, C;
    dd_sincos_small(p, &S, &C);  // |xi - alpha| <= 0.52 A <= 0.83
    dd_store(xS, N, j, S);
    dd_store(xC, N, j, C);
}

// out_c <- out_c / xi'  (the factor of (2.8)); fp64, or dd planar with plane size L
__global__ void k_mesh_scale_f64(int N, size_t total, const double* __restrict__ xE, double* __restrict__ out) {
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= total) return;
    out[e] /= xE[e & (size_t)(N - 1)];
}
__global__ void k_mesh_scale_dd(int N, size_t total, size_t L, const double* __restrict__ xE, double* __restrict__ out) {
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= total) return;
    const dd r = dd_div(dd{out[e], out[L + e]}, dd_load(xE, N, e & (size_t)(N - 1)));
    out[e] = r.hi;
    out[L + e] = r.lo;
}

int mesh_scale_out(sww_dtn_s* d, double* out, int nrhs, size_t L) {
    if (!d->mesh_on || nrhs <= 0) return SWW_OK;
    const size_t total = (size_t)d->N * nrhs;
    SWW_BEGIN(KC_OTHER, d->stream);
    if (d->prec == SWW_DD) k_mesh_scale_dd<<<(unsigned)((total + 255) / 256), 256, 0, d->stream>>>(d->N, total, L ? L : total, d->mesh.xE, out);
    else k_mesh_scale_f64<<<(unsigned)((total + 255) / 256), 256, 0, d->stream>>>(d->N, total, d->mesh.xE, out);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

// ------------------------------------------------------------------------------------------------ respacing
// xi(b) - x and xi'(b) at a dd parameter value b for the mesh (rho, where)
__device__ inline void mesh_xi_dd(dd A, int where, dd b, dd* xi, dd* E) {
    dd s1, c1, s2, c2;
    dd_sincos_any(b, &s1, &c1);
    s2 = dd_mul_d(dd_mul(s1, c1), 2.0);
    c2 = dd_sub(dd_sqr(c1), dd_sqr(s1));
    const dd a1 = where == 0 ? dd_half(A) : dd_neg(dd_half(A)), a2 = dd_neg(dd_ldexp(A, -3));
    *xi = dd_add(b, dd_add(dd_mul(a1, s1), dd_mul(dd_half(a2), s2)));
    *E = dd_add(dd_add_d(dd_mul(a1, c1), 1.0), dd_mul(a2, c2));
}

// beta_j = xi_old^{-1}(xi_new(alpha_j)), alpha_j = 2 pi j / Mn, by Newton's method in dd; sj = sin(Mo beta_j / 2)
__global__ void k_respace_nodes(int Mo, double rho_o, int where_o, int Mn, double rho_n, int where_n, double* __restrict__ beta /* dd planar 2 Mn */,
                                double* __restrict__ sj /* dd planar 2 Mn */) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= Mn) return;
    const dd An = mesh_A(rho_n), Ao = mesh_A(rho_o);
    const dd al = dd_div_d(dd_mul_d(dd_mul_d(dd_pi(), 2.0), (double)j), (double)Mn);
    dd x, e;
    mesh_xi_dd(An, where_n, al, &x, &e);
    dd b = x;
    for (int it = 0; it < 40; it++) {
        dd xb, eb;
        mesh_xi_dd(Ao, where_o, b, &xb, &eb);
        const dd step = dd_div(dd_sub(xb, x), eb);
        b = dd_sub(b, step);
        if (fabs(step.hi) < 1e-31) break;
    }
    dd_store(beta, Mn, j, b);
    dd s, c;
    dd_sincos_any(dd_mul_d(b, 0.5 * (double)Mo), &s, &c);
    sj[j] = s.hi;
    sj[Mn + j] = s.lo;
}

// R[j + m Mn] = D(beta_j - alpha_m), alpha_m = 2 pi m / Mo, D(t) = (1/Mo) sin(Mo t / 2) cot(t / 2) the periodic Dirichlet kernel of Mo
// (even) points with the Nyquist mode as a cosine; sin(Mo (beta_j - alpha_m)/2) = (-1)^m sin(Mo beta_j / 2).  D(0) = 1.
__global__ void k_respace_matrix(int Mo, int Mn, const double* __restrict__ beta, const double* __restrict__ sj, double* __restrict__ R) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x, m = blockIdx.y;
    if (j >= Mn) return;
    const dd am = dd_div_d(dd_mul_d(dd_mul_d(dd_pi(), 2.0), (double)m), (double)Mo);
    const dd t = dd_sub(dd_load(beta, Mn, j), am);
    double th = 0.5 * (t.hi + t.lo);
    // |t| below 1e-13: sin(Mo t/2) cot(t/2) / Mo = 1 - O((Mo t)^2)
    double v;
    if (fabs(th) < 1e-13) v = 1.0;
    else {
        const double sg = (m & 1) ? -1.0 : 1.0;
        v = sg * sj[j] / (tan(th) * (double)Mo);
    }
    R[(size_t)j + (size_t)m * Mn] = v;
}

// the same matrix in double-double (planar, plane size Mn Mo): cot(t/2) from the dd sine and cosine
__global__ void k_respace_matrix_dd(int Mo, int Mn, const double* __restrict__ beta, const double* __restrict__ sj, double* __restrict__ R) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x, m = blockIdx.y;
    if (j >= Mn) return;
    const dd am = dd_div_d(dd_mul_d(dd_mul_d(dd_pi(), 2.0), (double)m), (double)Mo);
    const dd th = dd_half(dd_sub(dd_load(beta, Mn, j), am));
    dd v{1.0, 0.0};
    if (fabs(th.hi) >= 1e-20) {   // below: 1 - O((Mo t)^2) = 1 in dd
        dd sn, cn;
        dd_sincos_any(th, &sn, &cn);
        v = dd_div_d(dd_div(dd_mul(dd_load(sj, Mn, j), cn), sn), (double)Mo);
        if (m & 1) v = dd_neg(v);
    }
    const size_t o = (size_t)j + (size_t)m * Mn;
    R[o] = v.hi;
    R[(size_t)Mn * Mo + o] = v.lo;
}
// out (Mn x ncol, planes Lout apart) = R (Mn x Mo, dd planar) y (Mo x ncol, planes Lin apart), one thread per output entry
__global__ void k_respace_apply_dd(int Mo, int Mn, int ncol, const double* __restrict__ R, const double* __restrict__ y, size_t Lin,
                                   double* __restrict__ out, size_t Lout) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x, c = blockIdx.y;
    if (j >= Mn) return;
    const size_t plane = (size_t)Mn * Mo;
    const double* yc = y + (size_t)c * Mo;
    dd acc[4] = {{0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}, {0.0, 0.0}};  // independent chains
    for (int m = 0; m < Mo; m += 4) {
#pragma unroll
        for (int q = 0; q < 4; q++) {
            const size_t o = (size_t)j + (size_t)(m + q) * Mn;
            acc[q] = dd_fma(dd{R[o], R[plane + o]}, dd{yc[m + q], yc[Lin + m + q]}, acc[q]);
        }
    }
    const dd r = dd_add(dd_add(acc[0], acc[1]), dd_add(acc[2], acc[3]));
    out[(size_t)c * Mn + j] = r.hi;
    out[Lout + (size_t)c * Mn + j] = r.lo;
}

// ------------------------------------------------------------------------------------------------ respacing without any allocation
// sww_respace_noalloc: the respacing of sww_state_respace for callers that cannot call cudaMalloc (CUDA graph capture, serving loops).
// The scratch of k_respace_nodes (beta_j and sin(Mo beta_j / 2), double-double planar: 4 Mn doubles) lives in a file-scope device
// array of fixed size; the interpolation matrix is never stored (its entries are formed where they are used).  Every GPU that loads
// the library holds the 128 KB until exit.  In host code `g_respace_scratch` is only a stand-in for the symbol: kernels get the
// device address that cudaGetSymbolAddress returned for the current device (respace_scratch_ptr below).
constexpr int RESPACE_NOALLOC_MAX = 4096;  // largest new mesh (SWW_RESPACE_NOALLOC_MAX of include/sww.h)
static __device__ __align__(256) double g_respace_scratch[4 * RESPACE_NOALLOC_MAX];

constexpr int RESPACE_MAX_DEVICES = 64;
static double* g_respace_scratch_ptr[RESPACE_MAX_DEVICES];  // per device: the array's device address, looked up once
static int respace_scratch_ptr(double** out) {
    int dev = 0;
    SWW_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= RESPACE_MAX_DEVICES) return SWW_EINVAL;
    if (!g_respace_scratch_ptr[dev]) {
        double* ptr = nullptr;
        SWW_CUDA(cudaGetSymbolAddress((void**)&ptr, g_respace_scratch));
        if (!ptr) return SWW_ECUDA;
        g_respace_scratch_ptr[dev] = ptr;
    }
    *out = g_respace_scratch_ptr[dev];
    return SWW_OK;
}

// out[j + c Mn] = sum_m D(beta_j - alpha_m) f[m + c Mo], the entries of k_respace_matrix formed on the fly (same arithmetic); a thread
// serves one new node j and up to four columns (the entries do not depend on the column); alpha_m goes through shared memory in
// chunks of 128 (double-double: a quotient per m, not per (j, m)).  grid: (ceil(Mn / 128), ceil(ncol / 4)), 128 threads.
__global__ void __launch_bounds__(128) k_respace_direct(int Mo, int Mn, int ncol, const double* __restrict__ beta, const double* __restrict__ sj,
                                                        const double* __restrict__ f, double* __restrict__ out) {
    __shared__ double a_hi[128], a_lo[128];
    const int j = blockIdx.x * 128 + threadIdx.x, c0 = blockIdx.y * 4;
    const int nc = min(4, ncol - c0);
    const bool on = j < Mn;
    const dd bj = on ? dd_load(beta, Mn, j) : dd{0.0, 0.0};
    const double sjj = on ? sj[j] : 0.0, rMo = (double)Mo;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
    for (int m0 = 0; m0 < Mo; m0 += 128) {
        __syncthreads();
        if (m0 + threadIdx.x < Mo) {
            const dd am = dd_div_d(dd_mul_d(dd_mul_d(dd_pi(), 2.0), (double)(m0 + threadIdx.x)), rMo);
            a_hi[threadIdx.x] = am.hi;
            a_lo[threadIdx.x] = am.lo;
        }
        __syncthreads();
        if (!on) continue;
        const int mn = min(128, Mo - m0);
        for (int q = 0; q < mn; q++) {
            const int m = m0 + q;
            const dd t = dd_sub(bj, dd{a_hi[q], a_lo[q]});
            const double th = 0.5 * (t.hi + t.lo);
            double v = 1.0;
            if (fabs(th) >= 1e-13) v = ((m & 1) ? -sjj : sjj) / (tan(th) * rMo);
            for (int c = 0; c < nc; c++) acc[c] = fma(v, f[(size_t)(c0 + c) * Mo + m], acc[c]);
        }
    }
    if (on)
        for (int c = 0; c < nc; c++) out[(size_t)(c0 + c) * Mn + j] = acc[c];
}

}  // namespace sww

extern "C" {

int sww_dtn_set_mesh(sww_dtn_t d, double rho, int where) {
    if (!d || !(rho > 0.0 && rho <= 1.0) || (where != 0 && where != 1)) return SWW_EINVAL;
    const int N = d->N;
    d->has_base = false;
    if (rho == 1.0) {  // the uniform mesh
        d->mesh_on = false;
        d->mesh_rho = 1.0;
        d->mesh_where = 0;
        return SWW_OK;
    }
    if (!d->mesh_buf) {
        SWW_CUDA(cudaMalloc(&d->mesh_buf, sizeof(double) * (8 * (size_t)N + 4)));
        d->mesh.coef = d->mesh_buf + 8 * (size_t)N;
        d->mesh.xE = d->mesh_buf;
        d->mesh.xE1 = d->mesh_buf + 2 * (size_t)N;
        d->mesh.xS = d->mesh_buf + 4 * (size_t)N;
        d->mesh.xC = d->mesh_buf + 6 * (size_t)N;
    }
    SWW_BEGIN(KC_OTHER, d->stream);
    k_mesh_tables<<<(N + 127) / 128, 128, 0, d->stream>>>(N, rho, where, d->tab->cs, d->tab->sn, d->mesh_buf, d->mesh_buf + 2 * (size_t)N,
                                                        d->mesh_buf + 4 * (size_t)N, d->mesh_buf + 6 * (size_t)N, d->mesh_buf + 8 * (size_t)N);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    const double A = 8.0 * (1.0 - rho) / (5.0 + 3.0 * rho);
    d->mesh_on = true;
    d->mesh_rho = rho;
    d->mesh_where = where;
    d->mesh_a1 = where == 0 ? 0.5 * A : -0.5 * A;
    d->mesh_a2 = -0.125 * A;
    return SWW_OK;
}

int sww_mesh_points(int N, double rho, int where, double* x) {
    if (!x || N < 1 || !(rho > 0.0 && rho <= 1.0) || (where != 0 && where != 1)) return SWW_EINVAL;
    const long double A = 8.0L * (1.0L - (long double)rho) / (5.0L + 3.0L * (long double)rho), a1 = where == 0 ? A / 2 : -A / 2, a2 = -A / 8;
    const long double two_pi = 6.283185307179586476925286766559L;
    for (int j = 0; j < N; j++) {
        const long double al = two_pi * j / N;
        x[j] = (double)(al + a1 * sinl(al) + a2 / 2 * sinl(2 * al));
    }
    return SWW_OK;
}

int sww_state_set_mesh(sww_state_t s, double rho, int where) {
    if (!s) return SWW_EINVAL;
    return sww_dtn_set_mesh(s->dtn, rho, where);
}

int sww_state_respace(sww_state_t dst, sww_state_t src) {
    if (!dst || !src || dst == src) return SWW_EINVAL;
    if (dst->prec != src->prec || dst->nc != src->nc) return SWW_EINVAL;
    const int Mo = src->N, Mn = dst->N, ncol = 2 + 2 * src->nc;
    const bool isdd = dst->prec == SWW_DD;
    const size_t rmul = isdd ? 2 : 1;
    cudaStream_t st = dst->stream;
    SWW_CUDA(cudaStreamSynchronize(src->stream));  // the source state is complete before it is read on dst's stream
    const sww_dtn_s *dn = dst->dtn, *ds = src->dtn;
    const double rho_o = ds->mesh_on ? ds->mesh_rho : 1.0, rho_n = dn->mesh_on ? dn->mesh_rho : 1.0;
    const int where_o = ds->mesh_on ? ds->mesh_where : 0, where_n = dn->mesh_on ? dn->mesh_where : 0;
    const bool cached = dst->rsp_R && dst->rsp_Mo == Mo && dst->rsp_rho_o == rho_o && dst->rsp_where_o == where_o && dst->rsp_rho_n == rho_n &&
                        dst->rsp_where_n == where_n;
    if (!cached) {  // the matrix depends on the two meshes only: a shooting iteration builds it once per pair of segments
        if (dst->rsp_R && dst->rsp_Mo != Mo) {
            SWW_CUDA(cudaStreamSynchronize(st));
            cudaFree(dst->rsp_R);
            dst->rsp_R = nullptr;
        }
        if (!dst->rsp_R && cudaMalloc(&dst->rsp_R, sizeof(double) * rmul * (size_t)Mn * Mo) != cudaSuccess) return SWW_ENOMEM;
        dst->rsp_Mo = 0;
        double* beta = nullptr;
        if (cudaMalloc(&beta, sizeof(double) * 4 * (size_t)Mn) != cudaSuccess) return SWW_ENOMEM;
        SWW_BEGIN(KC_OTHER, st);
        k_respace_nodes<<<(Mn + 63) / 64, 64, 0, st>>>(Mo, rho_o, where_o, Mn, rho_n, where_n, beta, beta + 2 * (size_t)Mn);
        SWW_LAUNCHED();
        SWW_BEGIN(KC_OTHER, st);
        if (isdd) k_respace_matrix_dd<<<dim3((Mn + 127) / 128, Mo), 128, 0, st>>>(Mo, Mn, beta, beta + 2 * (size_t)Mn, dst->rsp_R);
        else k_respace_matrix<<<dim3((Mn + 127) / 128, Mo), 128, 0, st>>>(Mo, Mn, beta, beta + 2 * (size_t)Mn, dst->rsp_R);
        SWW_LAUNCHED();
        const bool ok = cudaGetLastError() == cudaSuccess && cudaStreamSynchronize(st) == cudaSuccess;
        cudaFree(beta);
        if (!ok) return SWW_ECUDA;
        dst->rsp_Mo = Mo; dst->rsp_rho_o = rho_o; dst->rsp_where_o = where_o; dst->rsp_rho_n = rho_n; dst->rsp_where_n = where_n;
    }
    if (isdd) {
        if (Mo % 4 != 0) return SWW_EINVAL;
        SWW_BEGIN(KC_DDGEMM, st);
        k_respace_apply_dd<<<dim3((Mn + 127) / 128, ncol), 128, 0, st>>>(Mo, Mn, ncol, dst->rsp_R, src->y, src->L, dst->y, dst->L);
        SWW_LAUNCHED();
        SWW_CUDA(cudaGetLastError());
    } else {
        SWW_TRY(gemm_f64(st, Mn, ncol, Mo, 1.0, dst->rsp_R, Mn, src->y, Mo, 0.0, dst->y, Mn, ncol));
    }
    SWW_CUDA(cudaStreamSynchronize(st));
    dst->t = src->t;
    dst->dtn->has_base = false;
    return SWW_OK;
}

int sww_respace_noalloc(int Mo, double rho_o, int where_o, int Mn, double rho_n, int where_n, int ncol, const double* f, double* out, void* stream) {
    if (!f || !out || f == out || ncol < 1) return SWW_EINVAL;
    if (Mo < 4 || (Mo & 1) || Mo > 8192 || Mn < 1) return SWW_EINVAL;
    if (!(rho_o > 0.0 && rho_o <= 1.0) || !(rho_n > 0.0 && rho_n <= 1.0) || (where_o != 0 && where_o != 1) || (where_n != 0 && where_n != 1))
        return SWW_EINVAL;
    if (Mn > RESPACE_NOALLOC_MAX) {  // the fixed scratch holds 4 doubles per new node
        snprintf(g_cuda_err, sizeof(g_cuda_err), "sww_respace_noalloc: M_new = %d exceeds SWW_RESPACE_NOALLOC_MAX = %d (fixed device scratch)", Mn,
                 RESPACE_NOALLOC_MAX);
        return SWW_ETOOBIG;
    }
    double* scr = nullptr;
    SWW_TRY(respace_scratch_ptr(&scr));  // the first call on a device looks the address up; no allocation here or below
    cudaStream_t st = (cudaStream_t)stream;
    // beta (2 Mn) and sin(Mo beta / 2) (2 Mn) are written in full for j < Mn before they are read: nothing of an earlier call survives
    k_respace_nodes<<<(Mn + 63) / 64, 64, 0, st>>>(Mo, rho_o, where_o, Mn, rho_n, where_n, scr, scr + 2 * (size_t)Mn);
    ++g_launches;
    k_respace_direct<<<dim3((Mn + 127) / 128, (ncol + 3) / 4), 128, 0, st>>>(Mo, Mn, ncol, scr, scr + 2 * (size_t)Mn, f, out);
    ++g_launches;
    SWW_CUDA(cudaGetLastError());
    return SWW_OK;
}

}  // extern "C"
