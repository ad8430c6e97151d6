// tables.cu -- per-N constant tables: cos/sin(2 pi m/N), (1/2)cot(pi m/N), sin^2(pi m/N), differentiation circulant,
// FFT twiddles.  "(1/2)cot((alpha_i - alpha_j)/2) ... computed once and for all", PAPER.md:150 (section 2.2).
// Computed on the device in double-double, cached per (device, N) for the life of the process.
#include "common.cuh"
#include "dd.cuh"
#include <mutex>
#include <map>
#include <vector>

namespace sww {

unsigned long long g_launches = 0;
char g_cuda_err[256] = "";
int note_cuda(cudaError_t e, const char* where) {
    snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s", where, cudaGetErrorString(e));
    return SWW_ECUDA;
}

int sm_count() {
    static int sms[256] = {0};
    int dev = 0;
    cudaGetDevice(&dev);
    dev &= 255;
    if (!sms[dev]) {
        cudaDeviceGetAttribute(&sms[dev], cudaDevAttrMultiProcessorCount, dev);
        if (sms[dev] <= 0) sms[dev] = 148;
    }
    return sms[dev];
}

// ---- per-kernel-class timing (diagnostics; see common.cuh)
bool g_timing = false;
namespace {
struct TimedLaunch { cudaEvent_t e0, e1; int cls; };
std::vector<TimedLaunch> g_timed;       // event pairs recorded since the last sww_timing_read
std::vector<cudaEvent_t> g_event_pool;  // recycled events
cudaStream_t g_cur_stream = nullptr;
TimedLaunch g_cur;
bool g_cur_open = false;
cudaEvent_t take_event() {
    if (!g_event_pool.empty()) { cudaEvent_t e = g_event_pool.back(); g_event_pool.pop_back(); return e; }
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    return e;
}
}  // namespace
void timing_begin(int cls, cudaStream_t st) {
    g_cur.e0 = take_event();
    g_cur.e1 = take_event();
    g_cur.cls = cls;
    g_cur_stream = st;
    g_cur_open = true;
    cudaEventRecord(g_cur.e0, st);
}
void timing_end() {
    if (!g_cur_open) return;
    cudaEventRecord(g_cur.e1, g_cur_stream);
    g_timed.push_back(g_cur);
    g_cur_open = false;
}

__global__ void k_tables(int N, double* cs, double* sn, double* c0, double* s2, double* dc, double* dc2, double2* tw, double* filt, double* filt_dd) {
    int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= N) return;
    {
        const int ak = (2 * m <= N) ? m : N - m;          // |k| of DFT index m
        const double x = (double)ak / (double)(N / 2);
        const double x2 = x * x, x4 = x2 * x2, x8 = x4 * x4, x16 = x8 * x8, x32 = x16 * x16;
        filt[m] = exp(-36.0 * (x32 * x4));                 // (2.14)
        // the same in double-double (x is exact: a ratio of an integer and a power of two)
        const dd y2 = dd_sqr(dd{x, 0.0}), y4 = dd_sqr(y2), y8 = dd_sqr(y4), y16 = dd_sqr(y8), y32 = dd_sqr(y16);
        dd_store(filt_dd, N, m, dd_exp(dd_mul_d(dd_mul(y32, y4), -36.0)));
    }
    dd s, c;
    dd_sincos_2pi_frac(m, N, &s, &c);
    dd_store(cs, N, m, c);
    dd_store(sn, N, m, s);
    tw[m] = make_double2(c.hi, -s.hi);
    // half angle pi m / N = 2 pi m / (2N)
    dd sh, ch;
    dd_sincos_2pi_frac(m, 2LL * N, &sh, &ch);
    dd cot = (m == 0) ? dd{0.0, 0.0} : dd_half(dd_div(ch, sh));
    if (2 * m == N) cot = dd{0.0, 0.0};  // cot(pi/2) = 0 exactly
    dd_store(c0, N, m, cot);
    dd_store(s2, N, m, dd_sqr(sh));
    dd d = (m & 1) ? dd_neg(cot) : cot;  // (1/2)(-1)^m cot(pi m/N): Fourier differentiation matrix for even N (Nyquist -> 0, R4)
    dd_store(dc, N, m, d);
    // D(D .) as one circulant: symbol -k^2 for |k| < N/2 and 0 at the Nyquist mode (R4) = the textbook second-derivative matrix
    // (-(-1)^m / (2 sin^2(pi m/N)), -N^2/12 - 1/6 on the diagonal) minus its Nyquist term (1/N)(-(N/2)^2)(-1)^m.  The entry of
    // m = N/2 is stored halved: the node-prep kernel sums c2[m] (f_{i-m} + f_{i+m}) over m = 1 .. N/2 and meets that node twice.
    dd c2;
    if (m == 0) {
        c2 = dd_add_d(dd_neg(dd_add(dd_div_d(dd{(double)N * (double)N, 0.0}, 12.0), dd_div_d(dd{1.0, 0.0}, 6.0))), 0.25 * (double)N);
    } else {
        c2 = dd_sub(dd{0.25 * (double)N, 0.0}, dd_div(dd{0.5, 0.0}, dd_sqr(sh)));
        if (m & 1) c2 = dd_neg(c2);
        if (2 * m == N) c2 = dd_half(c2);
    }
    dd_store(dc2, N, m, c2);
}

static std::mutex g_tab_mu;
static std::map<std::pair<int, int>, Tables*> g_tabs;

int get_tables(int N, cudaStream_t st, const Tables** out) {
    int dev = 0;
    SWW_CUDA(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lk(g_tab_mu);
    auto key = std::make_pair(dev, N);
    auto it = g_tabs.find(key);
    if (it != g_tabs.end()) {
        *out = it->second;
        return SWW_OK;
    }
    Tables* t = new Tables();
    t->N = N;
    double* base = nullptr;
    // 7 dd tables of 2N doubles + N double2 + N doubles
    SWW_CUDA(cudaMalloc(&base, sizeof(double) * (size_t)N * 17));
    t->cs = base;
    t->sn = base + 2 * (size_t)N;
    t->c0 = base + 4 * (size_t)N;
    t->s2 = base + 6 * (size_t)N;
    t->dc = base + 8 * (size_t)N;
    t->tw = reinterpret_cast<double2*>(base + 10 * (size_t)N);
    t->filt = base + 12 * (size_t)N;
    t->filt_dd = base + 13 * (size_t)N;
    t->dc2 = base + 15 * (size_t)N;
    // the default stream orders this before any later stream work after the synchronize below
    SWW_BEGIN(KC_OTHER, st);
    k_tables<<<(N + 127) / 128, 128, 0, st>>>(N, t->cs, t->sn, t->c0, t->s2, t->dc, t->dc2, t->tw, t->filt, t->filt_dd);
    SWW_LAUNCHED();
    SWW_CUDA(cudaGetLastError());
    SWW_CUDA(cudaStreamSynchronize(st));
    g_tabs[key] = t;
    *out = t;
    return SWW_OK;
}

}  // namespace sww

extern "C" {
int sww_timing_enable(int on) {
    sww::g_timing = on != 0;
    return SWW_OK;
}
int sww_timing_read(double* ms, unsigned long long* launches, int nclass) {
    using namespace sww;
    if (!ms || !launches || nclass < KC_COUNT) return SWW_EINVAL;
    for (int c = 0; c < nclass; c++) { ms[c] = 0.0; launches[c] = 0; }
    int rc = SWW_OK;
    for (auto& t : g_timed) {
        float f = 0.f;
        if (cudaEventSynchronize(t.e1) != cudaSuccess || cudaEventElapsedTime(&f, t.e0, t.e1) != cudaSuccess) rc = SWW_ECUDA;
        ms[t.cls] += f;
        launches[t.cls]++;
        g_event_pool.push_back(t.e0);
        g_event_pool.push_back(t.e1);
    }
    g_timed.clear();
    return rc;
}
}
