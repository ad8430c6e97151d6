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
#include <new>
#include <cstring>

using namespace sww;

struct sww_shooter_s {
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
__global__ void k_shoot_out(int N, int n, int isdd, size_t L, double whi, double wlo, const double* __restrict__ y, const double* __restrict__ k0,
                            double* __restrict__ r, double* __restrict__ J) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    const int col = blockIdx.y;  // 0: r ; 1: J column 0 ; 2..n+1: J columns 1..n
    const dd w{whi, wlo};
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

// one shot through the stepper s (with_cols: s carries the n variational columns and J is wanted)
static int shoot_impl(sww_shooter_t S, sww_state_s* s, bool with_cols, const double* c, int nsteps, void* r, void* J, void* eta_T4, void* phi_T4) {
    const int N = S->N, n = S->n, isdd = S->prec == SWW_DD;
    cudaStream_t st = s->stream;
    SWW_CUDA(cudaMemcpyAsync(S->c_dev, c, sizeof(double) * (n + 1), cudaMemcpyHostToDevice, st));
    SWW_CUDA(cudaStreamSynchronize(st));  // c may be pageable host memory that the caller changes right after the call
    const Tables* tab = s->dtn->tab;
    const dim3 blk(128), grd((N + 127) / 128, with_cols ? n + 1 : 1);
    SWW_BEGIN(KC_OTHER, st);
    k_shoot_init<<<grd, blk, 0, st>>>(N, n, isdd, s->L, tab->cs, S->c_dev, s->y);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    s->t = 0.0;
    if (S->sdc) SWW_TRY(sww_sdc_advance(s, c[0] / (4.0 * nsteps), nsteps));
    else SWW_TRY(sww_rk_advance(s, c[0] / (4.0 * nsteps), nsteps));
    if (with_cols) SWW_TRY(rk_rhs(s, s->y, s->k));  // phi_t at T/4 (stage slot 0)
    // w = 1/sqrt(N), N = 2^p: a power of two, times 1/sqrt(2) (double-double) when p is odd
    int p = 0;
    while ((1 << p) < N) p++;
    double whi = ldexp(1.0, -(p / 2)), wlo = 0.0;
    if (p & 1) {
        whi = ldexp(0.70710678118654757, -(p / 2));
        wlo = ldexp(-4.8336466567264567e-17, -(p / 2));
    }
    const dim3 grd2((N + 127) / 128, with_cols ? n + 2 : 1);
    SWW_BEGIN(KC_OTHER, st);
    k_shoot_out<<<grd2, blk, 0, st>>>(N, n, isdd, s->L, whi, wlo, s->y, s->k, (double*)r, (double*)J);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return sww_state_read(s, eta_T4, phi_T4, nullptr, nullptr, nullptr);  // synchronises; the sticky status of the stepper's DtN handle
}

int sww_shoot(sww_shooter_t S, const double* c, int nsteps, void* r, void* J, void* eta_T4, void* phi_T4) {
    if (!S || !c || nsteps < 1 || !r || !J) return SWW_EINVAL;
    if (!(c[0] > 0.0)) return SWW_EINVAL;  // the period
    return shoot_impl(S, S->st, true, c, nsteps, r, J, eta_T4, phi_T4);
}

int sww_shoot_residual(sww_shooter_t S, const double* c, int nsteps, void* r) {
    if (!S || !c || nsteps < 1 || !r) return SWW_EINVAL;
    if (!(c[0] > 0.0)) return SWW_EINVAL;
    if (!S->st0) SWW_TRY(sww_state_create(S->N, S->h, S->g, S->prec, 0, S->zero, S->zero, nullptr, nullptr, S->flags, S->st->stream, &S->st0));
    S->st0->sigma = S->sigma;
    return shoot_impl(S, S->st0, false, c, nsteps, r, nullptr, nullptr, nullptr);
}

int sww_shooter_set_sigma(sww_shooter_t S, double sigma) {
    if (!S || !(sigma >= 0.0)) return SWW_EINVAL;
    S->sigma = sigma;
    S->st->sigma = sigma;
    if (S->st0) S->st0->sigma = sigma;
    return SWW_OK;
}

int sww_shooter_set_method(sww_shooter_t S, int method) {
    if (!S || (method != 0 && method != 1)) return SWW_EINVAL;
    S->sdc = method;
    return SWW_OK;
}

int sww_shooter_dims(sww_shooter_t S, int* N, int* n, int* is_dd) {
    if (!S) return SWW_EINVAL;
    if (N) *N = S->N;
    if (n) *n = S->n;
    if (is_dd) *is_dd = S->prec == SWW_DD;
    return SWW_OK;
}

int sww_shooter_destroy(sww_shooter_t S) {
    if (!S) return SWW_EINVAL;
    if (S->st) sww_state_destroy(S->st);
    if (S->st0) sww_state_destroy(S->st0);
    cudaFree(S->c_dev);
    cudaFree(S->zero);
    delete S;
    return SWW_OK;
}

}  // extern "C"
