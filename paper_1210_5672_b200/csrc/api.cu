// api.cu -- the C ABI of include/sww.h: handle management, right-hand-side formation (S3), the DtN apply (S4-S6), the base
// state (2.9) and the linearized DtN (B.1d),(B.2).  Product code; shares nothing with oracle/.
#include "common.cuh"
#include <algorithm>
#include "dd.cuh"
#include <new>
#include <cstring>

using namespace sww;

namespace sww {

static bool valid_N(int N) { return N >= 16 && N <= 8192 && (N & (N - 1)) == 0; }
static int pad64(int n) { return (n + 63) / 64 * 64; }

int ensure_workspace(sww_dtn_s* d, int nrhs) {
    int need = pad64(nrhs < 1 ? 1 : nrhs);
    Workspace& w = d->ws;
    if (need <= w.cap_cols) return SWW_OK;
    SWW_CUDA(cudaStreamSynchronize(d->stream));
    cudaFree(w.B); cudaFree(w.Gam); cudaFree(w.W); cudaFree(w.T); cudaFree(w.R); cudaFree(w.S);
    w = Workspace();
    size_t per = (size_t)d->N * need * sizeof(double) * (d->prec == SWW_DD ? 2 : 1);
    if (cudaMalloc(&w.B, per) != cudaSuccess || cudaMalloc(&w.Gam, per) != cudaSuccess || cudaMalloc(&w.W, per) != cudaSuccess ||
        cudaMalloc(&w.T, per) != cudaSuccess)
        return SWW_ENOMEM;
    if (d->prec == SWW_DD && cudaMalloc(&w.R, (size_t)d->N * need * sizeof(double)) != cudaSuccess) return SWW_ENOMEM;
    if (cudaMalloc(&w.S, (size_t)d->N * need * sizeof(double)) != cudaSuccess) return SWW_ENOMEM;
    SWW_CUDA(cudaMemsetAsync(w.B, 0, per, d->stream));
    SWW_CUDA(cudaMemsetAsync(w.Gam, 0, per, d->stream));
    SWW_CUDA(cudaMemsetAsync(w.W, 0, per, d->stream));
    SWW_CUDA(cudaMemsetAsync(w.T, 0, per, d->stream));
    w.cap_cols = need;
    return SWW_OK;
}

// ---- S3: right-hand sides --------------------------------------------------------------------------------------------
// plain apply: B = phi
// linearized : B_c = dphi_c - v deta_c  (B.1d);  T_c = u deta_c  (for the shape term of (B.2))
__global__ void k_rhs_lin_f64(int N, size_t total, const double* __restrict__ deta, const double* __restrict__ dphi,
                              const double* __restrict__ u, const double* __restrict__ v, double* __restrict__ B, double* __restrict__ T) {
    size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= total) return;
    int j = (int)(e & (size_t)(N - 1));
    double de = deta[e];
    B[e] = fma(-v[j], de, dphi[e]);
    T[e] = u[j] * de;
}

static int apply_f64(sww_dtn_s* d, const double* rhs_dev /* N x nrhs, or NULL when ws.B is already filled */, const double* Tcols,
                     int nrhs, double* out) {
    const int N = d->N;
    Workspace& w = d->ws;
    if (rhs_dev) SWW_CUDA(cudaMemcpyAsync(w.B, rhs_dev, sizeof(double) * (size_t)N * nrhs, cudaMemcpyDeviceToDevice, d->stream));
    SWW_TRY(run_solve(d, w.B, w.S, nrhs));                                       // S4: mu = A^{-1} b
    SWW_TRY(spectral_gamma_w(d, w.B, Tcols, w.Gam, out, nrhs, nrhs));           // S5: gamma = D mu ; out = |D| mu / 2 - D t
    if (nrhs <= 4 && N >= 128 && (size_t)d->bp_chunks * 4 >= 16)  // S6: out += G gamma   (2.8)
        SWW_TRY(gemv_few_f64(d->stream, N, nrhs, N, d->G, N, w.Gam, N, out, N, d->bp_part, d->mv_count));
    else
        SWW_TRY(gemm_f64(d->stream, N, nrhs, N, 1.0, d->G, N, w.Gam, N, 1.0, out, N, nrhs));
    return mesh_scale_out(d, out, nrhs, 0);  // the factor 1/|xi'| of (2.8) on a refined mesh
}


// eta_lo: the low words (double-double handles; nullptr = the N doubles behind eta)
int setup_surface(sww_dtn_s* d, const double* eta, const double* eta_lo) {
    const int N = d->N;
    d->has_base = false;
    SWW_CUDA(cudaMemcpyAsync(d->eta, eta, sizeof(double) * N, cudaMemcpyDeviceToDevice, d->stream));
    if (d->prec == SWW_F64) {
        SWW_CUDA(cudaMemsetAsync(d->eta + N, 0, sizeof(double) * N, d->stream));
        SWW_TRY(run_setup_f64(d));
    } else {
        SWW_CUDA(cudaMemcpyAsync(d->eta + N, eta_lo ? eta_lo : eta + N, sizeof(double) * N, cudaMemcpyDeviceToDevice, d->stream));
        SWW_TRY(run_setup_dd(d));
    }
    return run_lu(d);
}
static int do_setup(sww_dtn_s* d, const void* eta) { return setup_surface(d, (const double*)eta, nullptr); }

}  // namespace sww

extern "C" {

int sww_dtn_setup(const void* eta, int N, double h, int prec, void* stream, sww_dtn_t* out) {
    if (!eta || !out || !valid_N(N) || (prec != SWW_F64 && prec != SWW_DD) || !(h > 0.0)) return SWW_EINVAL;
    if (prec == SWW_DD && N > 4096) return SWW_EINVAL;  // the double-double spectral passes (ddpath.cu); include/sww.h states the limits
    sww_dtn_s* d = new (std::nothrow) sww_dtn_s();
    if (!d) return SWW_ENOMEM;
    memset(d, 0, sizeof(*d));
    new (&d->ws) Workspace();
    d->N = N;
    d->prec = prec;
    d->h = h;
    d->finite = !std::isinf(h);
    d->stream = (cudaStream_t)stream;
    int rc = get_tables(N, d->stream, &d->tab);
    if (rc) { delete d; return rc; }
    const size_t n2 = (size_t)N * N, mat = n2 * (prec == SWW_DD ? 2 : 1);
    const int nb = N < NB ? N : NB;
    bool ok = true;
    auto alloc = [&](double** p, size_t n) { if (ok && cudaMalloc(p, n * sizeof(double)) != cudaSuccess) ok = false; };
    alloc(&d->eta, 2 * N); alloc(&d->d1, 2 * N); alloc(&d->d2, 2 * N);
    alloc(&d->E, 2 * N); alloc(&d->Dm, 2 * N); alloc(&d->Sh, 2 * N); alloc(&d->Ch, 2 * N);
    alloc(&d->K, mat); alloc(&d->G, mat); alloc(&d->LU, n2); alloc(&d->invD, 3 * (size_t)N * nb);
    alloc(&d->bphi, 2 * N); alloc(&d->bW0, 2 * N); alloc(&d->bu, 2 * N); alloc(&d->bv, 2 * N); alloc(&d->tmp, 14 * (size_t)N);
    // column chunks of the dd base-state pass: enough CTAs to fill the chip at small N (4 columns per chunk at least)
    d->bp_chunks = std::max(1, std::min(N / 4, std::max(N / 32, 64)));
    alloc(&d->bp_part, (size_t)d->bp_chunks * 4 * N);
    if (ok && cudaMalloc(&d->status, sizeof(int)) != cudaSuccess) ok = false;
    if (ok && (cudaMalloc(&d->mv_count, sizeof(unsigned) * (N / 32 + 1)) != cudaSuccess ||
               cudaMemsetAsync(d->mv_count, 0, sizeof(unsigned) * (N / 32 + 1), d->stream) != cudaSuccess)) ok = false;
    if (!ok) { sww_dtn_destroy(d); return SWW_ENOMEM; }
    if (cudaMemsetAsync(d->status, 0, sizeof(int), d->stream) != cudaSuccess) { sww_dtn_destroy(d); return SWW_ECUDA; }
    rc = ensure_workspace(d, 64);
    if (!rc) rc = lu_alloc(d);
    if (!rc) rc = do_setup(d, eta);
    if (rc) { sww_dtn_destroy(d); return rc; }
    *out = d;
    return SWW_OK;
}

int sww_dtn_refactor(sww_dtn_t d, const void* eta) {
    if (!d || !eta) return SWW_EINVAL;
    return do_setup(d, eta);
}

int sww_dtn_apply(sww_dtn_t d, const void* phi, int nrhs, void* out) {
    if (!d || nrhs < 0) return SWW_EINVAL;
    if (nrhs == 0) return SWW_OK;  // an empty batch: the pointers are not looked at
    if (!phi || !out) return SWW_EINVAL;
    SWW_TRY(ensure_workspace(d, nrhs));
    if (d->prec == SWW_F64) return apply_f64(d, (const double*)phi, nullptr, nrhs, (double*)out);
    return dd_apply(d, (const double*)phi, false, nullptr, nrhs, (double*)out);
}

int sww_dtn_set_base(sww_dtn_t d, const void* phi0) {
    if (!d || !phi0) return SWW_EINVAL;
    SWW_TRY(ensure_workspace(d, 1));
    SWW_TRY(accurate_base(d, (const double*)phi0));
    d->has_base = true;
    return SWW_OK;
}

int sww_dtn_linearized_apply(sww_dtn_t d, const void* deta, const void* dphi, int nrhs, void* out) {
    if (!d || nrhs < 0) return SWW_EINVAL;
    if (!d->has_base) return SWW_ENOBASE;
    if (nrhs == 0) return SWW_OK;
    if (!deta || !dphi || !out) return SWW_EINVAL;
    SWW_TRY(ensure_workspace(d, nrhs));
    if (d->prec == SWW_DD) return dd_linearized(d, (const double*)deta, (const double*)dphi, nrhs, (double*)out);
    const int N = d->N;
    size_t total = (size_t)N * nrhs;
    SWW_BEGIN(KC_OTHER, d->stream);
    k_rhs_lin_f64<<<(unsigned)((total + 255) / 256), 256, 0, d->stream>>>(N, total, (const double*)deta, (const double*)dphi, d->bu, d->bv,
                                                                         d->ws.B, d->ws.T);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    return apply_f64(d, nullptr, d->ws.T, nrhs, (double*)out);
}

int sww_dtn_get(sww_dtn_t d, int which, void* dst) {
    if (!d || !dst) return SWW_EINVAL;
    const int N = d->N;
    const size_t mul = d->prec == SWW_DD ? 2 : 1;
    const double* src = nullptr;
    size_t n = 0;
    switch (which) {
        case 0: src = d->K; n = (size_t)N * N * mul; break;
        case 1: src = d->G; n = (size_t)N * N * mul; break;
        case 2: src = d->d1; n = N * mul; break;
        case 3: src = d->d2; n = N * mul; break;
        case 4: src = d->bphi; n = N * mul; break;
        case 5: src = d->bW0; n = N * mul; break;
        case 6: src = d->bu; n = N * mul; break;
        case 7: src = d->bv; n = N * mul; break;
        case 8: src = d->LU; n = (size_t)N * N; break;
        default: return SWW_EINVAL;
    }
    SWW_CUDA(cudaMemcpyAsync(dst, src, n * sizeof(double), cudaMemcpyDeviceToDevice, d->stream));
    return SWW_OK;
}

int sww_dtn_status(sww_dtn_t d) {
    if (!d) return SWW_EINVAL;
    int st = 0;
    SWW_CUDA(cudaMemcpyAsync(&st, d->status, sizeof(int), cudaMemcpyDeviceToHost, d->stream));
    SWW_CUDA(cudaStreamSynchronize(d->stream));
    return st;
}

int sww_dtn_destroy(sww_dtn_t d) {
    if (!d) return SWW_EINVAL;
    cudaStreamSynchronize(d->stream);
    double* ptrs[] = {d->eta, d->d1, d->d2, d->E, d->Dm, d->Sh, d->Ch, d->K, d->G, d->LU, d->invD, d->bphi, d->bW0, d->bu, d->bv, d->tmp, d->bp_part,
                      d->ws.B, d->ws.Gam, d->ws.W, d->ws.T, d->ws.R, d->ws.S};
    for (double* p : ptrs) cudaFree(p);
    cudaFree(d->mesh_buf);
    cudaFree(d->status);
    cudaFree(d->mv_count);
    cudaFree(d->lu_order);
    cudaFree(d->lu_flags);
    cudaFree(d->tr_flags);
    cudaFree(d->tr_scr);
    delete d;
    return SWW_OK;
}

const char* sww_strerror(int status) {
    switch (status) {
        case SWW_OK: return "ok";
        case SWW_EINVAL: return "invalid argument";
        case SWW_ENOMEM: return "out of memory";
        case SWW_ECUDA: return "CUDA runtime error";
        case SWW_EBOTTOM: return "surface touches the bottom (h + eta <= 0)";
        case SWW_ESINGULAR: return "pivot below guard in the unpivoted LU of I/2 + K";
        case SWW_ENOBASE: return "linearized apply before set_base";
        case SWW_ETOOBIG: return "size beyond the fixed scratch of a no-allocation entry point";
        default: return "unknown status";
    }
}
const char* sww_last_cuda_error(void) { return g_cuda_err; }
unsigned long long sww_launch_count(void) { return g_launches; }

// One cached context (handle + device staging buffers) for the HOST-pointer entry point: a caller that steps a surface calls
// this once per stage with the same N and precision, and creating a handle (about 150 MB of cudaMalloc at N = 2048) would cost
// ten times the computation.  The cache is replaced when N or the precision changes; sww_host_cache_clear() frees it.
namespace {
struct HostCtx {
    sww_dtn_t h = nullptr;
    int N = 0, prec = -1;
    size_t cap = 0;  // staging capacity in bytes of one batch buffer
    double *de = nullptr, *dp = nullptr, *dde = nullptr, *ddp = nullptr, *dout = nullptr;
    cudaStream_t copy_st = nullptr;  // the batch columns are uploaded here while setup + base state run on the compute stream
    cudaEvent_t in_ev = nullptr;
} g_host;
void host_ctx_free() {
    if (g_host.copy_st) cudaStreamSynchronize(g_host.copy_st);
    if (g_host.in_ev) cudaEventDestroy(g_host.in_ev);
    if (g_host.copy_st) cudaStreamDestroy(g_host.copy_st);
    if (g_host.h) sww_dtn_destroy(g_host.h);
    cudaFree(g_host.de); cudaFree(g_host.dp); cudaFree(g_host.dde); cudaFree(g_host.ddp); cudaFree(g_host.dout);
    g_host = HostCtx();
}
}  // namespace

int sww_host_cache_clear(void) {
    host_ctx_free();
    return SWW_OK;
}

int sww_dtn_linearized_host(const void* eta, const void* phi0, const void* deta, const void* dphi, void* out, int N, double h,
                            int prec, int nrhs) {
    if (!eta || !phi0 || !deta || !dphi || !out || nrhs < 1 || !valid_N(N) || (prec != SWW_F64 && prec != SWW_DD) || !(h > 0.0) ||
        (prec == SWW_DD && N > 4096))
        return SWW_EINVAL;
    const size_t mul = prec == SWW_DD ? 2 : 1, vec = sizeof(double) * N * mul, bat = vec * nrhs;
    cudaStream_t st = nullptr;
    HostCtx& c = g_host;
    if (c.N != N || c.prec != prec) host_ctx_free();
    if (!c.de) {
        if (cudaMalloc(&c.de, vec) || cudaMalloc(&c.dp, vec)) { host_ctx_free(); return SWW_ENOMEM; }
        c.N = N;
        c.prec = prec;
    }
    if (c.cap < bat) {
        cudaFree(c.dde); cudaFree(c.ddp); cudaFree(c.dout);
        c.dde = c.ddp = c.dout = nullptr;
        c.cap = 0;
        if (cudaMalloc(&c.dde, bat) || cudaMalloc(&c.ddp, bat) || cudaMalloc(&c.dout, bat)) { host_ctx_free(); return SWW_ENOMEM; }
        c.cap = bat;
    }
    if (!c.copy_st && (cudaStreamCreateWithFlags(&c.copy_st, cudaStreamNonBlocking) || cudaEventCreateWithFlags(&c.in_ev, cudaEventDisableTiming))) {
        host_ctx_free();
        return SWW_ECUDA;
    }
    // the surface and the base potential go first on the compute stream; the batch (the bulk of the bytes) is uploaded on a
    // second stream behind them and is only waited for where it is first read, after setup and the base state
    if (cudaMemcpyAsync(c.de, eta, vec, cudaMemcpyHostToDevice, st) || cudaMemcpyAsync(c.dp, phi0, vec, cudaMemcpyHostToDevice, st) ||
        cudaMemcpyAsync(c.dde, deta, bat, cudaMemcpyHostToDevice, c.copy_st) || cudaMemcpyAsync(c.ddp, dphi, bat, cudaMemcpyHostToDevice, c.copy_st) ||
        cudaEventRecord(c.in_ev, c.copy_st))
        return note_cuda(cudaGetLastError(), "host staging copies");
    int rc;
    if (!c.h) {
        rc = sww_dtn_setup(c.de, N, h, prec, st, &c.h);
    } else {
        c.h->h = h;  // a new depth is a new surface like any other
        c.h->finite = !std::isinf(h);
        rc = sww_dtn_refactor(c.h, c.de);
    }
    if (!rc) rc = sww_dtn_set_base(c.h, c.dp);
    if (cudaStreamWaitEvent(st, c.in_ev, 0) && !rc) rc = SWW_ECUDA;  // always waited for: the staging buffers must be idle on return
    if (!rc) rc = sww_dtn_linearized_apply(c.h, c.dde, c.ddp, nrhs, c.dout);
    if (!rc && cudaMemcpyAsync(out, c.dout, bat, cudaMemcpyDeviceToHost, st)) rc = SWW_ECUDA;
    if (!rc) rc = sww_dtn_status(c.h);  // synchronises
    else cudaStreamSynchronize(c.copy_st);
    if (rc) {  // a sticky device status (EBOTTOM, ESINGULAR) must not leak into the next call
        int keep = rc;
        host_ctx_free();
        return keep;
    }
    return SWW_OK;
}

}  // extern "C"
