// sdc_tables.cpp -- the constants of the SDC15 stepper: the s Radau IIa nodes on (0, 1] and the integration matrix
// S_mj = int_0^{c_m} l_j of the Lagrange basis on them, computed on the HOST in __float128 and returned as double-double pairs.
// Nodes: x = 1 and the roots of (P_s(x) - P_{s-1}(x)) / (x - 1), by Newton with deflation of the roots already found; matrix: the
// moment equations sum_j S_mj c_j^q = c_m^{q+1} / (q + 1), q = 0..s-1, solved by Gaussian elimination with partial pivoting.
// Product code (host side of rk.cu); shares nothing with oracle/.
#include <cmath>
#include <vector>

namespace sww {

typedef __float128 Q;

static void legendre_pair(int n, Q x, Q& pn, Q& pn1) {  // P_n(x), P_{n-1}(x)
    Q p0 = 1, p1 = x;
    for (int k = 2; k <= n; k++) {
        const Q p2 = ((2 * k - 1) * x * p1 - (k - 1) * p0) / k;
        p0 = p1;
        p1 = p2;
    }
    pn = (n == 0) ? (Q)1 : p1;
    pn1 = (n == 0) ? (Q)0 : p0;
}

static Q radau_f(int s, Q x) {
    Q a, b;
    legendre_pair(s, x, a, b);
    return a - b;
}

static void split(Q v, double& hi, double& lo) {
    hi = (double)v;
    lo = (double)(v - (Q)hi);
}

// c, dc (dc_m = c_m - c_{m-1}, c_0 = 0): s entries each; S: s x s row-major; all as (hi, lo)
int sdc_tables_host(int s, double* c_hi, double* c_lo, double* dc_hi, double* dc_lo, double* S_hi, double* S_lo) {
    if (s < 1 || s > 16) return -1;
    std::vector<Q> x;  // roots in (-1, 1), found one after another
    for (int i = 0; i < s - 1; i++) {
        Q z = -cosl((long double)(2 * i + 1) * 3.14159265358979323846L / (2 * s - 1));  // interlacing guesses
        for (int it = 0; it < 200; it++) {
            // g = f / ((x - 1) prod (x - x_r)): Newton on g through g'/g = f'/f - 1/(x-1) - sum 1/(x - x_r), f' by a centred difference
            const Q e = (Q)1e-12;
            const Q f = radau_f(s, z), df = (radau_f(s, z + e) - radau_f(s, z - e)) / (2 * e);
            Q corr = df / f - 1 / (z - 1);
            for (Q r : x) corr -= 1 / (z - r);
            const Q dz = 1 / corr;
            z -= dz;
            if ((dz < 0 ? -dz : dz) < (Q)1e-33) break;
        }
        // polish on f itself with the analytic derivative of P_s - P_{s-1}:  (1 - x^2) P_n' = n (P_{n-1} - x P_n)
        for (int it = 0; it < 4; it++) {
            Q ps, ps1, ps2, dummy;
            legendre_pair(s, z, ps, ps1);
            legendre_pair(s - 1, z, dummy, ps2);
            const Q dps = s * (ps1 - z * ps) / (1 - z * z), dps1 = (s - 1) * (ps2 - z * ps1) / (1 - z * z);
            z -= (ps - ps1) / (dps - dps1);
        }
        x.push_back(z);
    }
    // sort ascending, append x = 1
    for (size_t i = 0; i < x.size(); i++)
        for (size_t j = i + 1; j < x.size(); j++)
            if (x[j] < x[i]) std::swap(x[i], x[j]);
    std::vector<Q> c(s);
    for (int i = 0; i < s - 1; i++) c[i] = (x[i] + 1) / 2;
    c[s - 1] = 1;
    for (int i = 0; i + 1 < s; i++)
        if (!(c[i] > 0 && c[i] < c[i + 1])) return -2;
    // moment equations, one linear system with s right-hand sides:  V^T S^T = M,  V_jq = c_j^q,  M_qm = c_m^{q+1} / (q + 1)
    std::vector<Q> A((size_t)s * s), B((size_t)s * s);
    for (int q = 0; q < s; q++)
        for (int j = 0; j < s; j++) {
            Q p = 1, pm = c[j];
            for (int k = 0; k < q; k++) { p *= c[j]; pm *= c[j]; }
            A[(size_t)q * s + j] = p;               // row q: c_j^q
            B[(size_t)q * s + j] = pm / (q + 1);    // right-hand side for m = j
        }
    for (int k = 0; k < s; k++) {
        int piv = k;
        for (int i = k + 1; i < s; i++) {
            const Q a = A[(size_t)i * s + k] < 0 ? -A[(size_t)i * s + k] : A[(size_t)i * s + k];
            const Q b = A[(size_t)piv * s + k] < 0 ? -A[(size_t)piv * s + k] : A[(size_t)piv * s + k];
            if (a > b) piv = i;
        }
        for (int j = 0; j < s; j++) {
            std::swap(A[(size_t)k * s + j], A[(size_t)piv * s + j]);
            std::swap(B[(size_t)k * s + j], B[(size_t)piv * s + j]);
        }
        for (int i = k + 1; i < s; i++) {
            const Q l = A[(size_t)i * s + k] / A[(size_t)k * s + k];
            for (int j = k; j < s; j++) A[(size_t)i * s + j] -= l * A[(size_t)k * s + j];
            for (int j = 0; j < s; j++) B[(size_t)i * s + j] -= l * B[(size_t)k * s + j];
        }
    }
    for (int m = 0; m < s; m++)  // back substitution, column m of B -> row m of S
        for (int j = s - 1; j >= 0; j--) {
            Q v = B[(size_t)j * s + m];
            for (int k = j + 1; k < s; k++) v -= A[(size_t)j * s + k] * B[(size_t)k * s + m];
            B[(size_t)j * s + m] = v / A[(size_t)j * s + j];
        }
    for (int m = 0; m < s; m++) {
        split(c[m], c_hi[m], c_lo[m]);
        split(c[m] - (m ? c[m - 1] : (Q)0), dc_hi[m], dc_lo[m]);
        for (int j = 0; j < s; j++) split(B[(size_t)j * s + m], S_hi[m * s + j], S_lo[m * s + j]);
    }
    return 0;
}

}  // namespace sww
