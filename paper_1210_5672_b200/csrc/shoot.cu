// shoot.cu -- the shooting map of the overdetermined shooting method on the uniform mesh (section 3.1 / 3.3):
//   (3.15) PAPER.md:197-200  initial state from the unknowns c: eta^_k(0) = c_|k| (k even), phi^_k(0) = c_|k| (k odd), 1 <= |k| <= n,
//                            i.e. eta(x,0) = sum_{k even} 2 c_k cos kx, phi(x,0) = sum_{k odd} 2 c_k cos kx; T = c_0 (3.16)
//   (3.17) PAPER.md:208      r_i = phi(alpha_i, T/4) sqrt(1/N)
//   (3.31) PAPER.md:296      J_ik = d r_i / d c_k: columns k >= 1 are the variational solutions phidot_k(., T/4) sqrt(1/N) advanced
//                            together with q by (3.32); column 0 is phi_t(., T/4) sqrt(1/N) / 4 (R13)
// Everything runs on the device through the time stepper of rk.cu (one setup + batched linearized DtN per stage); this file
// only builds the initial state and scales the result.  Product code; shares nothing with oracle/.
#include "rk.cuh"
#include "dd.cuh"
#include "fft.cuh"
#include <new>
#include <vector>
#include <cstring>
#include <cmath>

using namespace sww;

constexpr int SHOOT_MAX_SEG = 8;
// one sub-interval of the mesh-refinement strategy of section 2.2; segment 0 runs on the shooter's own steppers
struct ShootSeg {
    int M, nsteps, where;
    double theta, rho;
    sww_state_t st, st0;  // the steppers of segments 1.. (with and without the columns; st0 created at the first residual-only shot)
};

struct sww_shooter_s {
    int nseg;             // 0: one uniform segment, the step count is the argument of sww_shoot
    ShootSeg seg[SHOOT_MAX_SEG];
    size_t zero_len;      // doubles behind `zero`
    int N, n, prec;
    double h, g, sigma;
    unsigned flags;
    int sdc;         // 1: advance by the SDC15 scheme (sww_sdc_advance) instead of RK8
    sww_state_t st;  // the stepper with the n variational columns
    sww_state_t st0; // the stepper without columns (residual-only shots), created at the first such shot
    double* c_dev;   // n + 1 unknowns
    double* zero;    // 2 N zeros (the flat state the stepper handle is created on)
};

namespace sww {

// 2 cos(k alpha_j) from the per-N table of cos(2 pi m / N) (double-double), with the phase k j reduced mod N exactly
__device__ __forceinline__ dd shoot_col(const double* cs, int N, int k, int j) {
    const int m = (int)(((long long)k * j) & (N - 1));
    return dd{2.0 * cs[m], 2.0 * cs[N + m]};
}

// state layout (rk.cuh): eta (N), phi (N), deta (N x n), dphi (N x n); double-double: the lo plane follows at + L
__global__ void k_shoot_init(int N, int n, int isdd, size_t L, const double* __restrict__ cs, const double* __restrict__ c, double* __restrict__ y) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    const int col = blockIdx.y;  // 0: eta and phi; k = 1..n: the columns d q0 / d c_k
    if (col == 0) {
        dd e{0.0, 0.0}, p{0.0, 0.0};
        for (int k = 1; k <= n; k++) {
            const dd t = dd_mul_d(shoot_col(cs, N, k, j), c[k]);
            if (k & 1) p = dd_add(p, t);
            else e = dd_add(e, t);
        }
        y[j] = e.hi;
        y[N + j] = p.hi;
        if (isdd) {
            y[L + j] = e.lo;
            y[L + N + j] = p.lo;
        }
    } else {
        const int k = col;
        const dd v = shoot_col(cs, N, k, j);
        const size_t oe = 2 * (size_t)N + (size_t)(k - 1) * N + j, op = oe + (size_t)N * n;
        const bool odd = k & 1;
        y[oe] = odd ? 0.0 : v.hi;
        y[op] = odd ? v.hi : 0.0;
        if (isdd) {
            y[L + oe] = odd ? 0.0 : v.lo;
            y[L + op] = odd ? v.lo : 0.0;
        }
    }
}

// r = phi w ; J[:, 0] = phi_t w / 4 ; J[:, k] = dphi_k w  (w = 1/sqrt(N) as a double-double).  Outputs: fp64, or double-double planar
// (r: hi block N, lo block N; J: hi block N (n+1), lo block N (n+1)).
// xE (refined last segment, dd planar; else nullptr): the weight is sqrt(E(alpha_j) / N) of (3.17)
__global__ void k_shoot_out(int N, int n, int isdd, size_t L, double whi, double wlo, const double* __restrict__ xE, const double* __restrict__ y,
                            const double* __restrict__ k0, double* __restrict__ r, double* __restrict__ J) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    const int col = blockIdx.y;  // 0: r ; 1: J column 0 ; 2..n+1: J columns 1..n
    dd w{whi, wlo};
    if (xE) w = isdd ? dd_sqrt(dd_div_d(dd{xE[j], xE[N + j]}, (double)N)) : dd{sqrt(xE[j] / (double)N), 0.0};
    size_t src;
    const double* base = y;
    double scale = 1.0;
    if (col == 0) src = (size_t)N + j;                       // phi
    else if (col == 1) { base = k0; src = (size_t)N + j; scale = 0.25; }   // phi_t
    else src = 2 * (size_t)N + (size_t)N * n + (size_t)(col - 2) * N + j;  // dphi_{k-1}
    dd v{base[src] * scale, isdd ? base[L + src] * scale : 0.0};
    v = dd_mul(v, w);
    double* dst = (col == 0) ? r : J;
    const size_t plane = (col == 0) ? (size_t)N : (size_t)N * (n + 1);
    const size_t o = (col == 0) ? (size_t)j : (size_t)(col - 1) * N + j;
    dst[o] = isdd ? v.hi : v.hi + v.lo;
    if (isdd) dst[plane + o] = v.lo;
}

// ------------------------------------------------------------------------------------------------ gradient of f by the adjoint system
// Section 3.2, (3.21)-(3.30): f = <(0, phi(T/4)), (0, phi(T/4))> / 2 with <a, b> = (1/2pi) int (eta_a eta_b + phi_a phi_b) dx
// (3.20); the adjoint solution q~ of (3.27), q~_s = DF(q(T/4 - s))^* q~ from q~(0) = (0, phi(T/4)), gives df/dq_0 = q~(T/4) (3.29) and
// df/dc_k = <q~(T/4), dq_0/dc_k> (3.30), df/dT = <(0, phi), (0, phi_t)> / 4 at T/4 (3.22).  Here the backward solve is the exact
// transpose of the forward Runge-Kutta recursion of the variational equation (the stage states Y_i of every step are kept, so no
// dense output is needed): with mu = F^* lambda_{n+1} (the filter after the step),
//     g_i = h b_i mu + h sum_{j>i} a_ji theta_j ,  theta_i = DF(Y_i)^* F^* g_i  (i = s..1),   lambda_n = mu + sum_i theta_i ,
// DF(Y)^* the right-hand side (B.6) of the adjoint system (sww_dtn_adjoint_rhs), F the filter (2.14) (self-adjoint on the uniform mesh;
// on a refined mesh F^* = E^{-1} F E in the inner product weighted by dx = E dalpha).
struct GradComb {
    int n;
    int idx[RK_S];
    double coef[RK_S];
    double cmu;
};
// out = cmu mu + sum_j coef_j theta[idx_j]   (vectors of 2N)
__global__ void k_grad_comb(size_t L, const double* __restrict__ mu, const double* __restrict__ theta, GradComb cb, double* __restrict__ out) {
    const size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= L) return;
    double v = cb.cmu * mu[q];
    for (int j = 0; j < cb.n; j++) v = fma(cb.coef[j], theta[(size_t)cb.idx[j] * L + q], v);
    out[q] = v;
}
// lambda (2N: eta~ | phi~) <- F^* lambda, one CTA
__global__ void __launch_bounds__(1024) k_grad_filter(int N, int logN, const double2* __restrict__ tw, const double* __restrict__ filt,
                                                      const double* __restrict__ xE, double* __restrict__ lam) {
    extern __shared__ __align__(16) double2 z[];
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const double e = xE ? xE[j] : 1.0;
        z[j] = make_double2(lam[j] * e, lam[N + j] * e);
    }
    __syncthreads();
    fft_dif(z, N, tw);
    const double rN = 1.0 / (double)N;
    for (int p = threadIdx.x; p < N; p += blockDim.x) {
        const double f = filt[(int)(__brev((unsigned)p) >> (32 - logN))] * rN;
        z[p] = make_double2(f * z[p].x, f * z[p].y);
    }
    __syncthreads();
    ifft_dit(z, N, tw);
    for (int j = threadIdx.x; j < N; j += blockDim.x) {
        const double re = xE ? 1.0 / xE[j] : 1.0;
        lam[j] = z[j].x * re;
        lam[N + j] = z[j].y * re;
    }
}
// out[0] = f = (1/2N) sum phi^2 E ; out[1] = df/dT = (1/4N) sum phi phi_t E ; lam <- (0, phi)   (3.21), (3.22), (3.26); one CTA
__global__ void __launch_bounds__(256) k_grad_start(int N, const double* __restrict__ y, const double* __restrict__ k0, const double* __restrict__ xE,
                                                    double* __restrict__ lam, double* __restrict__ out) {
    __shared__ double s0[256], s1[256];
    double a = 0.0, b = 0.0;
    for (int j = threadIdx.x; j < N; j += 256) {
        const double p = y[N + j], e = xE ? xE[j] : 1.0;
        a = fma(p * p, e, a);
        b = fma(p * k0[N + j], e, b);
        lam[j] = 0.0;
        lam[N + j] = p;
    }
    s0[threadIdx.x] = a;
    s1[threadIdx.x] = b;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) {
            s0[threadIdx.x] += s0[threadIdx.x + o];
            s1[threadIdx.x] += s1[threadIdx.x + o];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        out[0] = 0.5 * s0[0] / (double)N;
        out[1] = 0.25 * s1[0] / (double)N;
    }
}
// out[2 + k - 1] = df/dc_k = (1/N) sum_j lam_field(j) 2 cos(k alpha_j), field = eta~ for even k, phi~ for odd k ((3.15), (3.30));
// one CTA per k = 1..n.  The initial state lives on the uniform mesh.
__global__ void __launch_bounds__(256) k_grad_project(int N, const double* __restrict__ cs, const double* __restrict__ lam, double* __restrict__ out) {
    __shared__ double s0[256];
    const int k = blockIdx.x + 1;
    const double* f = (k & 1) ? lam + N : lam;
    double a = 0.0;
    for (int j = threadIdx.x; j < N; j += 256) a = fma(f[j], 2.0 * cs[(int)(((long long)k * j) & (N - 1))], a);
    s0[threadIdx.x] = a;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) s0[threadIdx.x] += s0[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) out[1 + k] = s0[0] / (double)N;
}

}  // namespace sww

extern "C" {

int sww_shooter_create(int N, int n, double h, double g, int prec, unsigned flags, void* stream, sww_shooter_t* out) {
    if (!out || n < 1 || N < 16 || 2 * n >= N) return SWW_EINVAL;  // modes 1..n must be resolved below the Nyquist mode
    sww_shooter_s* S = new (std::nothrow) sww_shooter_s();
    if (!S) return SWW_ENOMEM;
    memset(S, 0, sizeof(*S));
    S->N = N; S->n = n; S->prec = prec; S->h = h; S->g = g; S->flags = flags;
    const size_t mul = prec == SWW_DD ? 2 : 1;
    const size_t nz = mul * (size_t)N * n;  // the larger of the zero arrays the create call reads (deta, dphi)
    S->zero_len = nz;
    if (cudaMalloc(&S->c_dev, sizeof(double) * (n + 1)) != cudaSuccess || cudaMalloc(&S->zero, sizeof(double) * nz) != cudaSuccess) {
        sww_shooter_destroy(S);
        return SWW_ENOMEM;
    }
    cudaStream_t st = (cudaStream_t)stream;
    if (cudaMemsetAsync(S->zero, 0, sizeof(double) * nz, st) != cudaSuccess) {
        sww_shooter_destroy(S);
        return SWW_ECUDA;
    }
    // the stepper on the flat state of rest (validates N, h, prec and the stepper's size limits); every shot overwrites it
    int rc = sww_state_create(N, h, g, prec, n, S->zero, S->zero, S->zero, S->zero, flags, stream, &S->st);
    if (rc) {
        sww_shooter_destroy(S);
        return rc;
    }
    *out = S;
    return SWW_OK;
}

// the stepper of segment l, with or without the columns (those without are created at the first residual-only shot)
static int seg_state(sww_shooter_t S, int l, bool with_cols, sww_state_s** out) {
    sww_state_t* slot = l == 0 ? (with_cols ? &S->st : &S->st0) : (with_cols ? &S->seg[l].st : &S->seg[l].st0);
    if (!*slot) {
        const int M = l == 0 ? S->N : S->seg[l].M;
        SWW_TRY(sww_state_create(M, S->h, S->g, S->prec, with_cols ? S->n : 0, S->zero, S->zero, with_cols ? S->zero : nullptr,
                                 with_cols ? S->zero : nullptr, S->flags, S->st->stream, slot));
        if (l > 0) SWW_TRY(sww_state_set_mesh(*slot, S->seg[l].rho, S->seg[l].where));
    }
    (*slot)->sigma = S->sigma;
    *out = *slot;
    return SWW_OK;
}

static int advance(sww_shooter_t S, sww_state_s* s, double dt, int nsteps) {
    return S->sdc ? sww_sdc_advance(s, dt, nsteps) : sww_rk_advance(s, dt, nsteps);
}

// one shot (with_cols: the steppers carry the n variational columns and J is wanted)
static int shoot_impl(sww_shooter_t S, bool with_cols, const double* c, int nsteps, void* r, void* J, void* eta_T4, void* phi_T4) {
    const int n = S->n, isdd = S->prec == SWW_DD;
    sww_state_s* s = nullptr;
    SWW_TRY(seg_state(S, 0, with_cols, &s));
    cudaStream_t st = s->stream;
    SWW_CUDA(cudaMemcpyAsync(S->c_dev, c, sizeof(double) * (n + 1), cudaMemcpyHostToDevice, st));
    SWW_CUDA(cudaStreamSynchronize(st));  // c may be pageable host memory that the caller changes right after the call
    {
        const int N = S->N;
        const dim3 blk(128), grd((N + 127) / 128, with_cols ? n + 1 : 1);
        SWW_BEGIN(KC_OTHER, st);
        k_shoot_init<<<grd, blk, 0, st>>>(N, n, isdd, s->L, s->dtn->tab->cs, S->c_dev, s->y);
        SWW_LAUNCHED();
        SWW_CUDA(cudaGetLastError());
    }
    s->t = 0.0;
    if (S->nseg == 0) {
        SWW_TRY(advance(S, s, c[0] / (4.0 * nsteps), nsteps));
    } else {  // section 2.2: segment l takes nsteps_l steps over theta_l T/4 on its own mesh; respacing in between
        for (int l = 0; l < S->nseg; l++) {
            if (l > 0) {
                sww_state_s* nx = nullptr;
                SWW_TRY(seg_state(S, l, with_cols, &nx));
                SWW_TRY(sww_state_respace(nx, s));
                s = nx;
            }
            SWW_TRY(advance(S, s, S->seg[l].theta * c[0] / (4.0 * S->seg[l].nsteps), S->seg[l].nsteps));
        }
    }
    const int N = s->N;  // the residual count m = M_nu
    if (with_cols) SWW_TRY(rk_rhs(s, s->y, s->k));  // phi_t at T/4 (stage slot 0)
    // w = 1/sqrt(N), N = 2^p: a power of two, times 1/sqrt(2) (double-double) when p is odd
    int p = 0;
    while ((1 << p) < N) p++;
    double whi = ldexp(1.0, -(p / 2)), wlo = 0.0;
    if (p & 1) {
        whi = ldexp(0.70710678118654757, -(p / 2));
        wlo = ldexp(-4.8336466567264567e-17, -(p / 2));
    }
    const dim3 blk(128), grd2((N + 127) / 128, with_cols ? n + 2 : 1);
    SWW_BEGIN(KC_OTHER, st);
    k_shoot_out<<<grd2, blk, 0, st>>>(N, n, isdd, s->L, whi, wlo, s->dtn->mesh_on ? s->dtn->mesh.xE : nullptr, s->y, s->k, (double*)r, (double*)J);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return sww_state_read(s, eta_T4, phi_T4, nullptr, nullptr, nullptr);  // synchronises; the sticky status of the stepper's DtN handle
}

int sww_shoot(sww_shooter_t S, const double* c, int nsteps, void* r, void* J, void* eta_T4, void* phi_T4) {
    if (!S || !c || (S->nseg == 0 && nsteps < 1) || !r || !J) return SWW_EINVAL;
    if (!(c[0] > 0.0)) return SWW_EINVAL;  // the period
    return shoot_impl(S, true, c, nsteps, r, J, eta_T4, phi_T4);
}

int sww_shoot_residual(sww_shooter_t S, const double* c, int nsteps, void* r) {
    if (!S || !c || (S->nseg == 0 && nsteps < 1) || !r) return SWW_EINVAL;
    if (!(c[0] > 0.0)) return SWW_EINVAL;
    return shoot_impl(S, false, c, nsteps, r, nullptr, nullptr, nullptr);
}

int sww_shoot_gradient(sww_shooter_t S, const double* c, int nsteps, double* f, double* grad) {
    if (!S || !c || nsteps < 1 || !grad) return SWW_EINVAL;
    if (!(c[0] > 0.0)) return SWW_EINVAL;
    if (S->prec != SWW_F64 || S->nseg != 0 || S->sdc) return SWW_EINVAL;  // fp64, one uniform segment, the Runge-Kutta stepper
    const int N = S->N, n = S->n, logN = fft_ilog2(N);
    sww_state_s* s = nullptr;
    SWW_TRY(seg_state(S, 0, false, &s));
    cudaStream_t st = s->stream;
    sww_dtn_s* d = s->dtn;
    const Tables* tab = d->tab;
    const size_t V = 2 * (size_t)N;  // one vector (eta | phi)
    // work space: the stage tape, theta_1..theta_s, mu, g, lambda, the outputs
    double* buf = nullptr;
    const size_t ntape = (size_t)nsteps * RK_S * V, nwork = (RK_S + 4) * V + (size_t)n + 2;
    SWW_CUDA(cudaMalloc(&buf, sizeof(double) * (ntape + nwork)));
    double *tape = buf, *theta = buf + ntape, *mu = theta + RK_S * V, *gv = mu + V, *lam = gv + V, *scr = lam + V, *out = scr + V;
    int rc = SWW_OK;
    auto run = [&]() -> int {
        SWW_CUDA(cudaMemcpyAsync(S->c_dev, c, sizeof(double) * (n + 1), cudaMemcpyHostToDevice, st));
        SWW_CUDA(cudaStreamSynchronize(st));
        SWW_BEGIN(KC_OTHER, st);
        k_shoot_init<<<dim3((N + 127) / 128, 1), 128, 0, st>>>(N, n, 0, s->L, tab->cs, S->c_dev, s->y);
        SWW_LAUNCHED();
        SWW_CUDA(cudaGetLastError());
        s->t = 0.0;
        const double dt = c[0] / (4.0 * nsteps);
        s->tape = tape;
        s->tape_steps = nsteps;
        const int rf = sww_rk_advance(s, dt, nsteps);   // forward solve (2.1), stage states kept
        s->tape = nullptr;
        s->tape_steps = 0;
        SWW_TRY(rf);
        SWW_TRY(rk_rhs(s, s->y, s->k));                 // phi_t at T/4
        const double* xE = d->mesh_on ? d->mesh.xE : nullptr;
        SWW_BEGIN(KC_OTHER, st);
        k_grad_start<<<1, 256, 0, st>>>(N, s->y, s->k, xE, lam, out);
        SWW_LAUNCHED();
        SWW_CUDA(cudaGetLastError());
        static DeviceOnce attr_once;
        if (attr_once.first()) SWW_CUDA(cudaFuncSetAttribute(k_grad_filter, cudaFuncAttributeMaxDynamicSharedMemorySize, 8192 * 16));
        auto filter_adj = [&](double* v) -> int {
            if (!s->filter) return SWW_OK;
            SWW_BEGIN(KC_FFT, st);
            k_grad_filter<<<1, fft_threads(N), sizeof(double2) * (size_t)N, st>>>(N, logN, tab->tw, tab->filt, xE, v);
            SWW_LAUNCHED();
            SWW_CUDA(cudaGetLastError());
            return SWW_OK;
        };
        const unsigned blocks = (unsigned)((V + 255) / 256);
        for (int nn = nsteps - 1; nn >= 0; nn--) {       // the transposed recursion, step by step backward
            SWW_CUDA(cudaMemcpyAsync(mu, lam, sizeof(double) * V, cudaMemcpyDeviceToDevice, st));
            SWW_TRY(filter_adj(mu));
            bool used[RK_S];
            for (int i = RK_S - 1; i >= 0; i--) {
                GradComb cb;
                cb.n = 0;
                cb.cmu = dt * s->b[i];
                for (int j = i + 1; j < RK_S; j++)
                    if (s->a[j][i] != 0.0 && used[j]) {
                        cb.idx[cb.n] = j;
                        cb.coef[cb.n] = dt * s->a[j][i];
                        cb.n++;
                    }
                used[i] = cb.n > 0 || cb.cmu != 0.0;
                if (!used[i]) continue;                   // a stage nothing depends on contributes nothing
                SWW_BEGIN(KC_OTHER, st);
                k_grad_comb<<<blocks, 256, 0, st>>>(V, mu, theta, cb, gv);
                SWW_LAUNCHED();
                SWW_CUDA(cudaGetLastError());
                SWW_TRY(filter_adj(gv));
                const double* Y = tape + ((size_t)nn * RK_S + i) * V;
                SWW_TRY(sww_dtn_refactor(d, Y));
                SWW_TRY(sww_dtn_set_base(d, Y + N));
                SWW_TRY(sww_dtn_adjoint_rhs(d, gv, gv + N, 1, s->g, s->sigma, theta + (size_t)i * V, theta + (size_t)i * V + N));
            }
            GradComb cb;                                  // lambda_n = mu + sum_i theta_i
            cb.n = 0;
            cb.cmu = 1.0;
            for (int i = 0; i < RK_S; i++)
                if (used[i]) {
                    cb.idx[cb.n] = i;
                    cb.coef[cb.n] = 1.0;
                    cb.n++;
                }
            SWW_BEGIN(KC_OTHER, st);
            k_grad_comb<<<blocks, 256, 0, st>>>(V, mu, theta, cb, lam);
            SWW_LAUNCHED();
            SWW_CUDA(cudaGetLastError());
        }
        SWW_BEGIN(KC_OTHER, st);
        k_grad_project<<<n, 256, 0, st>>>(N, tab->cs, lam, out);
        SWW_LAUNCHED();
        SWW_CUDA(cudaGetLastError());
        std::vector<double> host((size_t)n + 2);
        SWW_CUDA(cudaMemcpyAsync(host.data(), out, sizeof(double) * (n + 2), cudaMemcpyDeviceToHost, st));
        SWW_TRY(sww_dtn_status(d));  // synchronises
        if (f) *f = host[0];
        for (int k = 0; k <= n; k++) grad[k] = host[1 + k];
        return SWW_OK;
    };
    rc = run();
    cudaStreamSynchronize(st);
    cudaFree(buf);
    return rc;
}

static void free_segments(sww_shooter_t S) {
    for (int l = 1; l < S->nseg; l++) {
        if (S->seg[l].st) sww_state_destroy(S->seg[l].st);
        if (S->seg[l].st0) sww_state_destroy(S->seg[l].st0);
        S->seg[l].st = S->seg[l].st0 = nullptr;
    }
    S->nseg = 0;
}

int sww_shooter_set_segments(sww_shooter_t S, int nu, const int* M, const double* theta, const double* rho, const int* where, const int* nsteps) {
    if (!S || nu < 0 || nu > SHOOT_MAX_SEG) return SWW_EINVAL;
    if (nu == 0) {
        free_segments(S);
        return SWW_OK;
    }
    if (!M || !theta || !rho || !where || !nsteps) return SWW_EINVAL;
    if (M[0] != S->N || rho[0] != 1.0) return SWW_EINVAL;  // the initial state (3.15) lives on the uniform mesh (rho_1 = 1)
    double sum = 0.0;
    size_t need = S->zero_len;
    for (int l = 0; l < nu; l++) {
        if (!(theta[l] > 0.0) || !(rho[l] > 0.0 && rho[l] <= 1.0) || (where[l] != 0 && where[l] != 1) || nsteps[l] < 1 || M[l] < 16) return SWW_EINVAL;
        sum += theta[l];
        const size_t nl = (S->prec == SWW_DD ? 2 : 1) * (size_t)M[l] * S->n;
        need = need > nl ? need : nl;
    }
    if (fabs(sum - 1.0) > 1e-12) return SWW_EINVAL;
    free_segments(S);
    if (need > S->zero_len) {
        SWW_CUDA(cudaStreamSynchronize(S->st->stream));
        cudaFree(S->zero);
        S->zero = nullptr;
        S->zero_len = 0;
        SWW_CUDA(cudaMalloc(&S->zero, sizeof(double) * need));
        SWW_CUDA(cudaMemsetAsync(S->zero, 0, sizeof(double) * need, S->st->stream));
        S->zero_len = need;
    }
    for (int l = 0; l < nu; l++) {
        S->seg[l].M = M[l]; S->seg[l].theta = theta[l]; S->seg[l].rho = rho[l]; S->seg[l].where = where[l]; S->seg[l].nsteps = nsteps[l];
        S->seg[l].st = S->seg[l].st0 = nullptr;
    }
    S->nseg = nu;
    for (int l = 1; l < nu; l++) {  // the steppers with the columns now (validates the sizes); those without at the first residual-only shot
        sww_state_s* s = nullptr;
        const int rc = seg_state(S, l, true, &s);
        if (rc) {
            free_segments(S);
            return rc;
        }
    }
    return SWW_OK;
}

int sww_shooter_set_sigma(sww_shooter_t S, double sigma) {
    if (!S || !(sigma >= 0.0)) return SWW_EINVAL;
    S->sigma = sigma;  // handed to every stepper at its next shot (seg_state)
    return SWW_OK;
}

int sww_shooter_set_method(sww_shooter_t S, int method) {
    if (!S || (method != 0 && method != 1)) return SWW_EINVAL;
    S->sdc = method;
    return SWW_OK;
}

int sww_shooter_dims(sww_shooter_t S, int* N, int* n, int* is_dd) {
    if (!S) return SWW_EINVAL;
    if (N) *N = S->nseg > 0 ? S->seg[S->nseg - 1].M : S->N;  // the number of residuals m = M_nu (3.17)
    if (n) *n = S->n;
    if (is_dd) *is_dd = S->prec == SWW_DD;
    return SWW_OK;
}

int sww_shooter_destroy(sww_shooter_t S) {
    if (!S) return SWW_EINVAL;
    free_segments(S);
    if (S->st) sww_state_destroy(S->st);
    if (S->st0) sww_state_destroy(S->st0);
    cudaFree(S->c_dev);
    cudaFree(S->zero);
    delete S;
    return SWW_OK;
}

}  // extern "C"
