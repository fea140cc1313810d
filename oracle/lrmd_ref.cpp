// lrmd_ref — the ORACLE for arXiv 1212.0262 (T. M. Rocha Filho, "Molecular dynamics for
// long-range interacting systems on Graphic Processing Units").
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
// bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code, header,
// constant table or helper with the CUDA path (paper_1212_0262_b200/csrc) and neither
// includes the other.
//
// What it is: a plain, serial (optionally OpenMP over the row index i only — every row sum
// keeps its serial j order, so results are bit-identical for any thread count), fp64
// restatement of what the paper's method computes.  The method is exact (it reaches the
// plain definition up to rounding order), so the oracle is the definition written out:
//
//   forces   f = -dH/dq of the three Hamiltonians, eq.(1) Ring
//            eq.(2) HMF, eq.(3) 2D self-gravity, summed over j != i in index order;
//   HMF      also through the mean-field identity PAPER.md:69-77 eqs.(5)-(7);
//   Ring     also through the per-particle sin/cos rewrite PAPER.md:97 eq.(9);
//   energies K = 1/2 sum p^2, V = the i<j double sum of eqs.(1)-(3), HMF also eq.(5);
//   step     Yoshida's 4th-order composition PAPER.md:48-50 eq.(4), 12-step listing PAPER.md:54-62.
//
// Readings of the paper taken here:
//   G1  eq.(8) prints f_ij with a PLUS sign; -dH/dtheta of eq.(1) has a MINUS sign.  The
//       Hamiltonian is the authority: f_i = -(1/(2 sqrt2 N)) sum_j sin(ti-tj)/(1-cos(ti-tj)+eps)^(3/2).
//   G2  listing step 11 prints f^(I); eq.(4)'s last factor acts at r(t+dt): the closing kick
//       uses the force computed in step 10.
//   G3  step 12 (truncated in the text) = reuse f(t+dt) as f^(I) of the next step: 3n+1 force
//       evaluations for n steps ("three force calculations").
//   G4  B0,B1,D0,D1 are not printed ("obtained in Ref. [33]"): Yoshida's triple-jump,
//       w1 = 1/(2-2^(1/3)), w0 = -2^(1/3)/(2-2^(1/3)); D0 = w1, D1 = w0, B0 = w1/2, B1 = (w0+w1)/2.
//   G5  the self term j = i is skipped explicitly (so eps = 0 is allowed when no two particles coincide).
//   G8  angles are never wrapped.
//
// Summation: every long sum (row sums over j, M, K, V, total momentum) is a Neumaier
// compensated sum, so the oracle's own rounding error stays ~1e-16 relative to sum|terms|
// at N = 5e7 (a naive serial sum would be ~1e-12, the size of the force tolerance).
//
// Pins (tests/test_oracle_*.py, -m "not gpu"): 50-digit mpmath derivative of the Hamiltonians,
// HMF pair sum vs identity, Ring eq.(8) vs eq.(9), regular-polygon closed forms, two-body
// closed forms (pendulum period 4K(k), circular orbit), 4th-order scaling, reversibility,
// momentum / angular momentum conservation, large-eps Ring -> HMF limit.
// Unpinned: the paper's Figs. 3-6 (images absent from the reference; "parity unpinned" for those).
//
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC (oracle/build.py).  No -ffast-math.

#include <cmath>
#include <cstddef>
#include <cstdint>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

enum Model { HMF = 0, RING = 1, GRAV2D = 2 };

// Neumaier's compensated summation.
struct Sum {
    double s = 0.0, c = 0.0;
    inline void add(double x) {
        const double t = s + x;
        if (std::fabs(s) >= std::fabs(x)) c += (s - t) + x;
        else                              c += (x - t) + s;
        s = t;
    }
    inline double value() const { return s + c; }
};

const double SQRT2 = std::sqrt(2.0);

// ---- pair terms f_ij (without the common prefactor), j != i -------------------------------

// HMF, -d/dtheta_i of (1/N)[1 - cos(ti - tj)] (eq.(2)):  -(1/N) sin(ti - tj)
inline double hmf_pair(double ti, double tj) { return std::sin(ti - tj); }

// Ring, eq.(8) PAPER.md:88 (sign per reading G1): sin(D) / (1 - cos(D) + eps)^(3/2)
inline double ring_pair_direct(double ti, double tj, double eps) {
    const double D = ti - tj;
    const double d = 1.0 - std::cos(D) + eps;
    return std::sin(D) / (d * std::sqrt(d));
}

// Ring, eq.(9): the same with per-particle sin/cos
inline double ring_pair_pre(double si, double ci, double sj, double cj, double eps) {
    const double num = si * cj - ci * sj;
    const double d = 1.0 - ci * cj - si * sj + eps;
    return num / (d * std::sqrt(d));
}

struct Ctx {
    int model;
    int64_t N;
    double eps;
    const double* q0;   // theta | x
    const double* q1;   // NULL  | y
};

// Force on particle i summed over all j != i in index order.  form: see lrmd_ref_forces.
// If A0/A1 are non-null also returns sum_j |f_ij| (with the prefactor).
inline void row_force(const Ctx& c, int form, int64_t i, const double* sn, const double* cs,
                      double* f0, double* f1, double* A0, double* A1) {
    const int64_t N = c.N;
    Sum a, b, aa, ab;
    if (c.model == HMF) {
        const double ti = c.q0[i];
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            const double t = hmf_pair(ti, c.q0[j]);
            a.add(t); aa.add(std::fabs(t));
        }
        const double pre = -1.0 / (double)N;
        *f0 = pre * a.value();
        if (A0) *A0 = std::fabs(pre) * aa.value();
    } else if (c.model == RING) {
        const double ti = c.q0[i];
        if (form == 0) {
            for (int64_t j = 0; j < N; ++j) {
                if (j == i) continue;
                const double t = ring_pair_direct(ti, c.q0[j], c.eps);
                a.add(t); aa.add(std::fabs(t));
            }
        } else {
            const double si = sn[i], ci = cs[i];
            for (int64_t j = 0; j < N; ++j) {
                if (j == i) continue;
                const double t = ring_pair_pre(si, ci, sn[j], cs[j], c.eps);
                a.add(t); aa.add(std::fabs(t));
            }
        }
        const double pre = -1.0 / (2.0 * SQRT2 * (double)N);
        *f0 = pre * a.value();
        if (A0) *A0 = std::fabs(pre) * aa.value();
    } else {
        // 2D: -d/dr_i of (1/N) log(|ri-rj|^2 + eps) (eq.(3)) = -(2/N)(ri-rj)/(|ri-rj|^2+eps)
        const double xi = c.q0[i], yi = c.q1[i];
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            const double dx = xi - c.q0[j], dy = yi - c.q1[j];
            const double r2 = dx * dx + dy * dy + c.eps;
            const double tx = dx / r2, ty = dy / r2;
            a.add(tx); b.add(ty); aa.add(std::fabs(tx)); ab.add(std::fabs(ty));
        }
        const double pre = -2.0 / (double)N;
        *f0 = pre * a.value();
        *f1 = pre * b.value();
        if (A0) *A0 = std::fabs(pre) * aa.value();
        if (A1) *A1 = std::fabs(pre) * ab.value();
    }
}

// HMF magnetisation, eq.(7)
inline void magnetisation(int64_t N, const double* th, double* Mx, double* My) {
    Sum sx, sy;
    for (int64_t i = 0; i < N; ++i) { sx.add(std::cos(th[i])); sy.add(std::sin(th[i])); }
    *Mx = sx.value() / (double)N;
    *My = sy.value() / (double)N;
}

int check(int model, int64_t N, double eps, const double* q0, const double* q1) {
    if (model < 0 || model > 2 || N < 1 || !q0) return -1;
    if (model == GRAV2D && !q1) return -1;
    if (model != HMF && !(eps >= 0.0)) return -1;
    return 0;
}

void set_threads(int nthreads) {
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
}

// rows == NULL: all rows 0..N-1 (nrows ignored).
int forces_impl(int model, int64_t N, double eps, const double* q0, const double* q1,
                const int64_t* rows, int64_t nrows, double* f0, double* f1,
                double* A0, double* A1, int form, int nthreads) {
    if (check(model, N, eps, q0, q1) || !f0 || (model == GRAV2D && !f1)) return -1;
    const int64_t R = rows ? nrows : N;
    Ctx c{model, N, eps, q0, q1};
    if (model == HMF && form == 0) {
        // eq.(6) PAPER.md:73 with eq.(7)
        double Mx, My;
        magnetisation(N, q0, &Mx, &My);
        double aSx = 0, aSy = 0;
        if (A0) {   // O(N) upper bound S_i >= A_i used at sizes where the pair sum is impossible
            Sum ac, as;
            for (int64_t j = 0; j < N; ++j) { ac.add(std::fabs(std::cos(q0[j]))); as.add(std::fabs(std::sin(q0[j]))); }
            aSx = ac.value() / (double)N; aSy = as.value() / (double)N;
        }
        for (int64_t r = 0; r < R; ++r) {
            const int64_t i = rows ? rows[r] : r;
            if (i < 0 || i >= N) return -1;
            const double ci = std::cos(q0[i]), si = std::sin(q0[i]);
            f0[r] = ci * My - si * Mx;
            if (A0) A0[r] = std::fabs(ci) * aSy + std::fabs(si) * aSx;
        }
        return 0;
    }
    std::vector<double> sn, cs;
    if (model == RING && form != 0) {
        sn.resize((size_t)N); cs.resize((size_t)N);
        for (int64_t j = 0; j < N; ++j) { sn[(size_t)j] = std::sin(q0[j]); cs[(size_t)j] = std::cos(q0[j]); }
    }
    for (int64_t r = 0; r < R; ++r) {
        const int64_t i = rows ? rows[r] : r;
        if (i < 0 || i >= N) return -1;
    }
    set_threads(nthreads);
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t r = 0; r < R; ++r) {
        const int64_t i = rows ? rows[r] : r;
        double d0 = 0, d1 = 0, a0 = 0, a1 = 0;
        row_force(c, form, i, sn.data(), cs.data(), &d0, &d1, A0 ? &a0 : nullptr, A1 ? &a1 : nullptr);
        f0[r] = d0;
        if (model == GRAV2D) f1[r] = d1;
        if (A0) A0[r] = a0;
        if (A1 && model == GRAV2D) A1[r] = a1;
    }
    return 0;
}

}  // namespace

extern "C" {

// Yoshida coefficients, reading G4.  out = {B0, B1, D0, D1}.
void lrmd_ref_coefficients(double* out) {
    const double cb = std::cbrt(2.0);
    const double w1 = 1.0 / (2.0 - cb);
    const double w0 = -cb / (2.0 - cb);
    out[0] = 0.5 * w1;
    out[1] = 0.5 * (w0 + w1);
    out[2] = w1;
    out[3] = w0;
}

// Forces on all N particles.  Host pointers.  q = (theta, NULL) or (x, y); f = (f, NULL) or (fx, fy).
// form: HMF   0 = mean-field identity eqs.(6)-(7), 1 = pair sum of eq.(2)
//       RING  0 = direct eq.(8),                   1 = precomputed sin/cos eq.(9)
//       2D    ignored
// nthreads: OpenMP threads over i (<= 0: runtime default); the result does not depend on it.
int lrmd_ref_forces(int model, int64_t N, double eps, const double* q0, const double* q1,
                    double* f0, double* f1, int form, int nthreads) {
    return forces_impl(model, N, eps, q0, q1, nullptr, 0, f0, f1, nullptr, nullptr, form, nthreads);
}

// Forces on the sampled rows only (each against all N).  Outputs have length nrows.
int lrmd_ref_forces_rows(int model, int64_t N, double eps, const double* q0, const double* q1,
                         const int64_t* rows, int64_t nrows, double* f0, double* f1,
                         int form, int nthreads) {
    if (!rows || nrows < 0) return -1;
    return forces_impl(model, N, eps, q0, q1, rows, nrows, f0, f1, nullptr, nullptr, form, nthreads);
}

// Forces and A_i = sum_{j != i} |f_ij| (the scale of the force tolerance) on rows (NULL = all).
// HMF form 0 returns the O(N) bound S_i = |cos ti| <|sin|> + |sin ti| <|cos|> >= A_i instead.
int lrmd_ref_abs_force_sums(int model, int64_t N, double eps, const double* q0, const double* q1,
                            const int64_t* rows, int64_t nrows, double* f0, double* f1,
                            double* A0, double* A1, int form, int nthreads) {
    if (!A0 || (model == GRAV2D && !A1)) return -1;
    return forces_impl(model, N, eps, q0, q1, rows, nrows, f0, f1, A0, A1, form, nthreads);
}

// out4 = {K, V, a, b}; HMF (a,b) = (Mx,My); RING (sum p, 0); 2D (sum px, sum py).
// out_abs (may be NULL) = {sum of |terms| of K, sum of |terms| of V} for tolerances.
// form: HMF 0 = V from eq.(5), 1 = V from the i<j pair sum of eq.(2); others: pair sum.
int lrmd_ref_energy(int model, int64_t N, double eps, const double* q0, const double* q1,
                    const double* p0, const double* p1, double* out4, double* out_abs,
                    int form, int nthreads) {
    if (check(model, N, eps, q0, q1) || !p0 || (model == GRAV2D && !p1) || !out4) return -1;
    Sum k, ka, pa, pb;
    for (int64_t i = 0; i < N; ++i) {
        double e = p0[i] * p0[i];
        pa.add(p0[i]);
        if (model == GRAV2D) { e += p1[i] * p1[i]; pb.add(p1[i]); }
        k.add(e);
    }
    const double K = 0.5 * k.value();
    double V = 0.0, Vabs = 0.0, a = pa.value(), b = pb.value();
    if (model == HMF) {
        magnetisation(N, q0, &a, &b);
    }
    if (model == HMF && form == 0) {
        V = 0.5 * (double)N * (1.0 - a * a - b * b);       // eq.(5)
        Vabs = 0.5 * (double)N;
    } else {
        std::vector<double> row((size_t)N, 0.0), rowabs((size_t)N, 0.0);
        set_threads(nthreads);
#pragma omp parallel for schedule(dynamic, 16)
        for (int64_t i = 0; i < N; ++i) {
            Sum s, sa;
            for (int64_t j = i + 1; j < N; ++j) {
                double t;
                if (model == HMF) {
                    t = 1.0 - std::cos(q0[i] - q0[j]);
                } else if (model == RING) {
                    t = 1.0 / (SQRT2 * std::sqrt(1.0 - std::cos(q0[i] - q0[j]) + eps));
                } else {
                    const double dx = q0[i] - q0[j], dy = q1[i] - q1[j];
                    t = std::log(dx * dx + dy * dy + eps);
                }
                s.add(t); sa.add(std::fabs(t));
            }
            row[(size_t)i] = s.value(); rowabs[(size_t)i] = sa.value();
        }
        Sum v, va;
        for (int64_t i = 0; i < N; ++i) { v.add(row[(size_t)i]); va.add(rowabs[(size_t)i]); }
        const double pre = (model == RING ? -1.0 : 1.0) / (double)N;
        V = pre * v.value();
        Vabs = va.value() / (double)N;
    }
    out4[0] = K; out4[1] = V; out4[2] = a; out4[3] = b;
    if (out_abs) { out_abs[0] = K; out_abs[1] = Vabs; }
    return 0;
}

// n steps of the 4th-order scheme, PAPER.md:54-62 under readings G2-G4, in place.
// f0/f1: the force array.  force_valid != 0: on entry it holds f(q) (reused as f^(I), G3);
// otherwise it is computed first (listing step 1).  On return it holds f(q(t + n dt)).
int lrmd_ref_step(int model, int64_t N, double eps, double* q0, double* q1, double* p0, double* p1,
                  double* f0, double* f1, int force_valid, int64_t n, double dt, int form, int nthreads) {
    if (check(model, N, eps, q0, q1) || !p0 || !f0 || n < 0) return -1;
    const bool two = (model == GRAV2D);
    if (two && (!p1 || !f1)) return -1;
    double co[4];
    lrmd_ref_coefficients(co);
    const double B[3] = {co[0], co[1], co[1]};   // B0, B1, B1
    const double D[3] = {co[2], co[3], co[2]};   // D0, D1, D0
    if (!force_valid) {                                           // step 1
        if (lrmd_ref_forces(model, N, eps, q0, q1, f0, f1, form, nthreads)) return -1;
    }
    for (int64_t s = 0; s < n; ++s) {
        for (int k = 0; k < 3; ++k) {
            const double b = B[k] * dt, d = D[k] * dt;
            for (int64_t i = 0; i < N; ++i) {
                p0[i] += b * f0[i];                               // steps 2, 5, 8
                q0[i] += d * p0[i];                               // steps 3, 6, 9
                if (two) { p1[i] += b * f1[i]; q1[i] += d * p1[i]; }
            }
            if (lrmd_ref_forces(model, N, eps, q0, q1, f0, f1, form, nthreads)) return -1;   // steps 4, 7, 10
        }
        const double b = B[0] * dt;
        for (int64_t i = 0; i < N; ++i) {                         // step 11 (G2: force of step 10)
            p0[i] += b * f0[i];
            if (two) p1[i] += b * f1[i];
        }
    }                                                             // step 12 (G3): f is reused
    return 0;
}

int lrmd_ref_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
