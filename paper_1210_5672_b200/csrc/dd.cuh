// dd.cuh -- double-double ("quadruple precision") arithmetic on the CUDA cores by error-free transformations.
// The algorithms are the classical ones (Dekker 1971 two-product via FMA, Knuth two-sum, Bailey-style dd add/mul/div);
// written here from their published definitions.  Product code; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>

namespace sww {

struct dd {
    double hi, lo;
};

__host__ __device__ __forceinline__ dd make_dd(double hi, double lo = 0.0) { return dd{hi, lo}; }

#ifdef __CUDA_ARCH__
#define SWW_ADD(a, b) __dadd_rn((a), (b))
#define SWW_SUB(a, b) __dsub_rn((a), (b))
#define SWW_MUL(a, b) __dmul_rn((a), (b))
#define SWW_FMA(a, b, c) __fma_rn((a), (b), (c))
#else
#define SWW_ADD(a, b) ((a) + (b))
#define SWW_SUB(a, b) ((a) - (b))
#define SWW_MUL(a, b) ((a) * (b))
#define SWW_FMA(a, b, c) fma((a), (b), (c))
#endif

// s + e = a + b exactly (6 flops)
__device__ __forceinline__ dd two_sum(double a, double b) {
    double s = SWW_ADD(a, b);
    double bb = SWW_SUB(s, a);
    double e = SWW_ADD(SWW_SUB(a, SWW_SUB(s, bb)), SWW_SUB(b, bb));
    return dd{s, e};
}
// requires |a| >= |b| (3 flops)
__device__ __forceinline__ dd quick_two_sum(double a, double b) {
    double s = SWW_ADD(a, b);
    double e = SWW_SUB(b, SWW_SUB(s, a));
    return dd{s, e};
}
// p + e = a * b exactly (2 flops)
__device__ __forceinline__ dd two_prod(double a, double b) {
    double p = SWW_MUL(a, b);
    double e = SWW_FMA(a, b, -p);
    return dd{p, e};
}

__device__ __forceinline__ dd dd_neg(dd a) { return dd{-a.hi, -a.lo}; }

// accurate dd + dd (20 flops)
__device__ __forceinline__ dd dd_add(dd a, dd b) {
    dd s = two_sum(a.hi, b.hi);
    dd t = two_sum(a.lo, b.lo);
    s.lo = SWW_ADD(s.lo, t.hi);
    s = quick_two_sum(s.hi, s.lo);
    s.lo = SWW_ADD(s.lo, t.lo);
    return quick_two_sum(s.hi, s.lo);
}
__device__ __forceinline__ dd dd_sub(dd a, dd b) { return dd_add(a, dd_neg(b)); }
__device__ __forceinline__ dd dd_add_d(dd a, double b) {
    dd s = two_sum(a.hi, b);
    s.lo = SWW_ADD(s.lo, a.lo);
    return quick_two_sum(s.hi, s.lo);
}
// dd * dd (9 flops with FMA)
__device__ __forceinline__ dd dd_mul(dd a, dd b) {
    dd p = two_prod(a.hi, b.hi);
    p.lo = SWW_FMA(a.hi, b.lo, p.lo);
    p.lo = SWW_FMA(a.lo, b.hi, p.lo);
    return quick_two_sum(p.hi, p.lo);
}
__device__ __forceinline__ dd dd_mul_d(dd a, double b) {
    dd p = two_prod(a.hi, b);
    p.lo = SWW_FMA(a.lo, b, p.lo);
    return quick_two_sum(p.hi, p.lo);
}
__device__ __forceinline__ dd dd_sqr(dd a) {
    dd p = two_prod(a.hi, a.hi);
    p.lo = SWW_FMA(SWW_MUL(2.0, a.hi), a.lo, p.lo);
    return quick_two_sum(p.hi, p.lo);
}
// c + a*b, dd accumulate (the inner operation of the dd GEMM / residual kernels): 2 + 2 + 6 + 1 + 3 = 14 flops
__device__ __forceinline__ dd dd_fma(dd a, dd b, dd c) {
    dd p = two_prod(a.hi, b.hi);
    p.lo = SWW_FMA(a.hi, b.lo, p.lo);
    p.lo = SWW_FMA(a.lo, b.hi, p.lo);
    dd s = two_sum(c.hi, p.hi);
    s.lo = SWW_ADD(s.lo, SWW_ADD(c.lo, p.lo));
    return quick_two_sum(s.hi, s.lo);
}
// The same accumulation without the renormalisation: c.hi + c.lo += a * b with c.hi the running two-sum of the high products and
// c.lo the plain fp64 sum of every error term (12 flops instead of 15).  c is NOT a normalised dd afterwards: |c.lo| grows by up to an
// ulp of c.hi per call, so the caller renormalises with dd_renorm every few dozen calls (and before c is used as a dd number).
__device__ __forceinline__ void dd_fma_lazy(dd a, dd b, dd& c) {
    const double p = SWW_MUL(a.hi, b.hi);
    double pe = SWW_FMA(a.hi, b.hi, -p);
    pe = SWW_FMA(a.hi, b.lo, pe);
    pe = SWW_FMA(a.lo, b.hi, pe);
    const double t = SWW_ADD(c.hi, p);
    const double bb = SWW_SUB(t, c.hi);
    const double e = SWW_ADD(SWW_SUB(c.hi, SWW_SUB(t, bb)), SWW_SUB(p, bb));
    c.lo = SWW_ADD(c.lo, SWW_ADD(e, pe));
    c.hi = t;
}
__device__ __forceinline__ dd dd_renorm(dd c) { return two_sum(c.hi, c.lo); }  // no assumption on |c.lo| against |c.hi|
// dd / dd by three quotient digits
__device__ __forceinline__ dd dd_div(dd a, dd b) {
    double q1 = a.hi / b.hi;
    dd r = dd_sub(a, dd_mul_d(b, q1));
    double q2 = r.hi / b.hi;
    r = dd_sub(r, dd_mul_d(b, q2));
    double q3 = r.hi / b.hi;
    dd q = quick_two_sum(q1, q2);
    return dd_add_d(q, q3);
}
__device__ __forceinline__ dd dd_div_d(dd a, double b) { return dd_div(a, dd{b, 0.0}); }
// sqrt(a), a > 0: the fp64 root x corrected by (a - x^2) / (2 x) (Karp-Markstein), the square taken error-free
__device__ __forceinline__ dd dd_sqrt(dd a) {
    const double x = sqrt(a.hi);
    const dd r = dd_sub(a, two_prod(x, x));
    return quick_two_sum(x, r.hi / (2.0 * x));
}
// fp64 reciprocal of a normal, well-scaled number: MUFU seed (2^-20) + two Newton steps (within an ulp), no slow path
// (|x| far from 0, inf, denormals)
__device__ __forceinline__ double rcp_normal(double x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    double e = SWW_FMA(-x, r, 1.0);
    r = SWW_FMA(r, e, r);
    e = SWW_FMA(-x, r, 1.0);
    r = SWW_FMA(r, e, r);
    return r;
}
// dd / dd in the hot loops (one kernel entry = two of these): two quotient digits from ONE fp64 reciprocal of b.hi.
// q1 = a.hi rb is within a few ulp of a/b; the remainder a - b q1 is formed exactly up to O(eps^2 |a|); q2 = r rb restores the
// low word: relative error ~ 1e-31 (the three-digit dd_div above, ~10x the instructions, is kept for the O(N) table setup).
__device__ __forceinline__ dd dd_div_rb(dd a, dd b, double rb) {
    const double q1 = SWW_MUL(a.hi, rb);
    const dd p = two_prod(b.hi, q1);
    double r = SWW_SUB(SWW_SUB(a.hi, p.hi), p.lo);  // a.hi - p.hi is exact (q1 b.hi is within a few ulp of a.hi)
    r = SWW_ADD(r, SWW_FMA(-b.lo, q1, a.lo));
    const double q2 = SWW_MUL(r, rb);
    return quick_two_sum(q1, q2);
}
__device__ __forceinline__ dd dd_div_fast(dd a, dd b) { return dd_div_rb(a, b, rcp_normal(b.hi)); }
// sinh, cosh of a small dd argument by the Taylor recurrences with the divisions replaced by dd reciprocals rc[m] =
// 1 / (m (m + 1)), m = 1..30 (hi at rc[m], lo at rc[32 + m]); the number of terms follows |x| (the last term kept is < 2^-110
// relative).  |x| < 0.5.
__device__ __forceinline__ void dd_sinhcosh_tab(dd x, const double* rc, dd* sh, dd* ch) {
    const dd x2 = dd_sqr(x);
    const int nt = (x2.hi < 1e-4) ? 6 : (x2.hi < 1e-2) ? 9 : 15;
    dd ts = x, tc = dd{1.0, 0.0}, ss = x, cc = dd{1.0, 0.0};
    for (int n = 1; n <= nt; n++) {
        tc = dd_mul(dd_mul(tc, x2), dd{rc[2 * n - 1], rc[32 + 2 * n - 1]});
        ts = dd_mul(dd_mul(ts, x2), dd{rc[2 * n], rc[32 + 2 * n]});
        cc = dd_add(cc, tc);
        ss = dd_add(ss, ts);
    }
    *sh = ss;
    *ch = cc;
}
__device__ __forceinline__ dd dd_from_diff(double a, double b) { return two_sum(a, -b); }  // exact a - b
__device__ __forceinline__ dd dd_ldexp(dd a, int e) { return dd{ldexp(a.hi, e), ldexp(a.lo, e)}; }
__device__ __forceinline__ dd dd_half(dd a) { return dd{0.5 * a.hi, 0.5 * a.lo}; }

// planar load/store: element idx of an array with L logical elements
__device__ __forceinline__ dd dd_load(const double* p, size_t L, size_t idx) { return dd{p[idx], p[L + idx]}; }
__device__ __forceinline__ void dd_store(double* p, size_t L, size_t idx, dd v) {
    p[idx] = v.hi;
    p[L + idx] = v.lo;
}

// ------------------------------------------------------------------ elementary functions (O(N) calls per setup only)
__device__ __forceinline__ dd dd_pi() { return dd{3.141592653589793116e+00, 1.224646799147353207e-16}; }
__device__ __forceinline__ dd dd_ln2() { return dd{6.931471805599452862e-01, 2.319046813846299558e-17}; }

// sin and cos of a dd angle |x| <= pi/4 + small, Taylor series summed until terms drop below 2^-115
__device__ inline void dd_sincos_small(dd x, dd* s, dd* c) {
    dd x2 = dd_sqr(x);
    dd ts = x, tc = dd{1.0, 0.0};
    dd ss = x, cc = dd{1.0, 0.0};
    for (int n = 1; n <= 16; n++) {
        // cos term: tc *= -x2 / ((2n-1)(2n)) ; sin term: ts *= -x2 / ((2n)(2n+1))
        tc = dd_neg(dd_div_d(dd_mul(tc, x2), (double)((2 * n - 1) * (2 * n))));
        ts = dd_neg(dd_div_d(dd_mul(ts, x2), (double)((2 * n) * (2 * n + 1))));
        cc = dd_add(cc, tc);
        ss = dd_add(ss, ts);
    }
    *s = ss;
    *c = cc;
}

// cos, sin(2 pi m / M) in dd with the angle reduced EXACTLY in integer arithmetic to [0, pi/4]
__device__ inline void dd_sincos_2pi_frac(long long m, long long M, dd* s, dd* c) {
    long long t = 4 * (m % M);
    long long quad = t / M, r = t - quad * M;  // angle = quad*pi/2 + (pi/2) r/M
    bool swap = false;
    if (2 * r > M) {
        r = M - r;
        swap = true;
    }
    dd ss, cc;
    if (r == 0) {
        ss = dd{0.0, 0.0};
        cc = dd{1.0, 0.0};
    } else {
        dd phi = dd_div_d(dd_mul_d(dd_half(dd_pi()), (double)r), (double)M);
        dd_sincos_small(phi, &ss, &cc);
        if (2 * r == M) cc = ss;
    }
    if (swap) {
        dd tmp = cc;
        cc = ss;
        ss = tmp;
    }
    switch (quad) {
        case 0: *c = cc; *s = ss; break;
        case 1: *c = dd_neg(ss); *s = cc; break;
        case 2: *c = dd_neg(cc); *s = dd_neg(ss); break;
        default: *c = ss; *s = dd_neg(cc); break;
    }
}

// exp of a dd argument, |x| < 700: x = k ln2 + r, |r| <= ln2/2, plain Taylor series in r (no squaring), scaled by 2^k
__device__ inline dd dd_exp(dd x) {
    double kf = rint(x.hi * 1.4426950408889634074);
    dd r = dd_sub(x, dd_mul_d(dd_ln2(), kf));
    dd term = dd{1.0, 0.0}, sum = dd{1.0, 0.0};
    for (int n = 1; n <= 27; n++) {
        term = dd_div_d(dd_mul(term, r), (double)n);
        sum = dd_add(sum, term);
    }
    return dd_ldexp(sum, (int)kf);
}
// expm1 for dd: series without the leading 1 when |x| is small (keeps relative accuracy), else exp(x) - 1
__device__ inline dd dd_expm1(dd x) {
    if (fabs(x.hi) < 0.34) {
        dd term = x, sum = x;
        for (int n = 2; n <= 27; n++) {
            term = dd_div_d(dd_mul(term, x), (double)n);
            sum = dd_add(sum, term);
        }
        return sum;
    }
    return dd_add_d(dd_exp(x), -1.0);
}
// sinh, cosh of a dd argument: odd/even Taylor series for |x| < 0.5 (relative accuracy for small x), else from exp
__device__ inline void dd_sinhcosh(dd x, dd* sh, dd* ch) {
    if (fabs(x.hi) < 0.5) {
        dd x2 = dd_sqr(x);
        dd ts = x, tc = dd{1.0, 0.0}, ss = x, cc = dd{1.0, 0.0};
        for (int n = 1; n <= 15; n++) {
            tc = dd_div_d(dd_mul(tc, x2), (double)((2 * n - 1) * (2 * n)));
            ts = dd_div_d(dd_mul(ts, x2), (double)((2 * n) * (2 * n + 1)));
            cc = dd_add(cc, tc);
            ss = dd_add(ss, ts);
        }
        *sh = ss;
        *ch = cc;
        return;
    }
    dd e = dd_exp(x);
    dd ei = dd_div(dd{1.0, 0.0}, e);
    *sh = dd_half(dd_sub(e, ei));
    *ch = dd_half(dd_add(e, ei));
}

// warp-wide dd sum (all lanes receive the total)
__device__ __forceinline__ dd dd_warp_sum(dd v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        dd w;
        w.hi = __shfl_xor_sync(0xffffffffu, v.hi, o);
        w.lo = __shfl_xor_sync(0xffffffffu, v.lo, o);
        v = dd_add(v, w);
    }
    return v;
}

}  // namespace sww
