// pp_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, obviously-correct CPU oracle for the direct particle-particle (PP) gravity path of
// Khrapov, Khoperskov & Khoperskov (2018), written from /root/reference/PAPER.md only.  It shares no code,
// header, table or helper with the CUDA library (paper_1803_01190_b200/csrc) and must never be imported,
// linked or executed by the product path: only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may use it.
//
// What it computes, and where the paper defines it:
//   oracle_forces*      eq. (1)-(2): a_i = sum_{j!=i} -G m_j (r_i-r_j) / |r_i-r_j+delta|^3 with
//                       |r_i-r_j+delta| = sqrt(dx^2+dy^2+dz^2+delta^2)  (reading R1), and
//                       the matching potential Phi_i = -G sum_{j!=i} m_j / |r_i-r_j+delta| whose gradient is eq. (2).
//   oracle_kdk_paper    eqs. (5)-(7), literally: predictor velocity, drift with the mean velocity,
//                       force recomputation, corrector.  One gravity solve per step.
//   oracle_kdk_halfkick the algebraically identical half-kick / drift / half-kick form (reading R4);
//                       exists only so that a test can show the two forms agree to round-off.
//   oracle_invariants   eqs. (8)-(10): E = K + W, P, L (all three components; the paper's L is
//                       L_z), plus centre of mass (Fig. 6) and total mass.  W carries the MINUS sign
//                       and excludes j == i (reading R3: the '+' and the j=i terms of eq. (8) are garbles).
//
// Arithmetic: IEEE double for every pair quantity; each per-particle running sum is a Neumaier (compensated)
// sum, sequential in j = 0..N-1, so the result does not depend on the thread count (threads split i only).
// The *_ld variants do the same in x87 long double with plain sums and exist to validate the compensated
// double version against something more precise (tests/test_oracle_pins.py).
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/oracle.py).  No -ffast-math: it would
// delete the compensation terms.
//
// Parity pins (tests/test_oracle_*.py, all CPU): P1 3-4-5 / 5-12-13 two-body values, P2 polygons, P3 antisymmetry,
// P4 a = -grad Phi, P5 softened circular binary, P6 Kepler period/energy/eccentricity + 2nd-order convergence,
// P7 time reversibility, P8 exact P and L conservation, P9 brute force N<=8 in exact rational arithmetic.
// No function in this file is "parity unpinned".

#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// Neumaier's improved Kahan-Babuska sum: s carries the running sum, c the accumulated low-order parts.
struct NSum {
    double s = 0.0, c = 0.0;
    inline void add(double x) {
        double t = s + x;
        if (std::fabs(s) >= std::fabs(x)) c += (s - t) + x;
        else                              c += (x - t) + s;
        s = t;
    }
    inline double value() const { return s + c; }
};

inline int clamp_threads(int nthreads) {
#ifdef _OPENMP
    if (nthreads <= 0) return omp_get_max_threads();
    return nthreads;
#else
    (void)nthreads;
    return 1;
#endif
}

// eq. (1)-(2) for one particle i (index into pos/mass).
inline void forces_one(const double* pos, const double* mass, int64_t N, double G, double delta,
                       int64_t i, double* a3, double* phi) {
    const double xi = pos[3 * i + 0], yi = pos[3 * i + 1], zi = pos[3 * i + 2];
    const double d2 = delta * delta;
    NSum ax, ay, az, ph;
    for (int64_t j = 0; j < N; ++j) {
        if (j == i) continue;                       // sum over j != i, eq. (1)
        const double dx = xi - pos[3 * j + 0];      // r_i - r_j
        const double dy = yi - pos[3 * j + 1];
        const double dz = zi - pos[3 * j + 2];
        const double r2 = dx * dx + dy * dy + dz * dz + d2;   // |r_i - r_j + delta|^2
        const double r = std::sqrt(r2);
        const double inv_r3 = 1.0 / (r2 * r);
        const double mj = mass[j];
        ax.add(-mj * dx * inv_r3);                  // eq. (2) without G
        ay.add(-mj * dy * inv_r3);
        az.add(-mj * dz * inv_r3);
        ph.add(-mj / r);
    }
    a3[0] = G * ax.value();
    a3[1] = G * ay.value();
    a3[2] = G * az.value();
    if (phi) *phi = G * ph.value();
}

inline void forces_one_ld(const double* pos, const double* mass, int64_t N, double G, double delta,
                          int64_t i, double* a3, double* phi) {
    const long double xi = pos[3 * i + 0], yi = pos[3 * i + 1], zi = pos[3 * i + 2];
    const long double d2 = (long double)delta * (long double)delta;
    long double ax = 0, ay = 0, az = 0, ph = 0;
    for (int64_t j = 0; j < N; ++j) {
        if (j == i) continue;
        const long double dx = xi - (long double)pos[3 * j + 0];
        const long double dy = yi - (long double)pos[3 * j + 1];
        const long double dz = zi - (long double)pos[3 * j + 2];
        const long double r2 = dx * dx + dy * dy + dz * dz + d2;
        const long double r = sqrtl(r2);
        const long double inv_r3 = 1.0L / (r2 * r);
        const long double mj = mass[j];
        ax -= mj * dx * inv_r3;
        ay -= mj * dy * inv_r3;
        az -= mj * dz * inv_r3;
        ph -= mj / r;
    }
    a3[0] = (double)((long double)G * ax);
    a3[1] = (double)((long double)G * ay);
    a3[2] = (double)((long double)G * az);
    if (phi) *phi = (double)((long double)G * ph);
}

void forces_all(const double* pos, const double* mass, int64_t N, double G, double delta,
                double* acc, double* pot, int nthreads) {
    const int nt = clamp_threads(nthreads);
    (void)nt;
#pragma omp parallel for schedule(dynamic, 16) num_threads(nt)
    for (int64_t i = 0; i < N; ++i) forces_one(pos, mass, N, G, delta, i, acc + 3 * i, pot ? pot + i : nullptr);
}

}  // namespace

extern "C" {

// Accelerations (and optionally potentials) of the particles listed in idx[0..n_idx) (idx == NULL: all N, then
// n_idx is ignored).  acc is [n,3], pot is [n] or NULL.  nthreads <= 0: all cores; 1: single-threaded.
void oracle_forces(const double* pos, const double* mass, int64_t N, double G, double delta,
                   const int64_t* idx, int64_t n_idx, double* acc, double* pot, int nthreads) {
    if (!idx) { forces_all(pos, mass, N, G, delta, acc, pot, nthreads); return; }
    const int nt = clamp_threads(nthreads);
    (void)nt;
#pragma omp parallel for schedule(dynamic, 4) num_threads(nt)
    for (int64_t k = 0; k < n_idx; ++k)
        forces_one(pos, mass, N, G, delta, idx[k], acc + 3 * k, pot ? pot + k : nullptr);
}

// Same contract, x87 long double pair arithmetic and sums (validation of the compensated-double version).
void oracle_forces_ld(const double* pos, const double* mass, int64_t N, double G, double delta,
                      const int64_t* idx, int64_t n_idx, double* acc, double* pot, int nthreads) {
    const int nt = clamp_threads(nthreads);
    (void)nt;
    const int64_t n = idx ? n_idx : N;
#pragma omp parallel for schedule(dynamic, 4) num_threads(nt)
    for (int64_t k = 0; k < n; ++k)
        forces_one_ld(pos, mass, N, G, delta, idx ? idx[k] : k, acc + 3 * k, pot ? pot + k : nullptr);
}

// eqs. (5)-(7) literally.  acc holds a(t) on entry if acc_valid != 0 (else it is computed
// first) and a(t + nsteps*dt) on exit: "a gravity solver ... only once at each time step".
// Returns the number of force evaluations performed.
int64_t oracle_kdk_paper(double* pos, double* vel, const double* mass, double* acc, int64_t N, double dt,
                         int64_t nsteps, double G, double delta, int acc_valid, int nthreads) {
    int64_t nforce = 0;
    if (!acc_valid) { forces_all(pos, mass, N, G, delta, acc, nullptr, nthreads); ++nforce; }
    std::vector<double> vtilde((size_t)(3 * N));
    for (int64_t s = 0; s < nsteps; ++s) {
        for (int64_t k = 0; k < 3 * N; ++k) vtilde[k] = vel[k] + dt * acc[k];                   // (5) predictor
        for (int64_t k = 0; k < 3 * N; ++k) pos[k] = pos[k] + (dt / 2.0) * (vtilde[k] + vel[k]); // (6) drift
        forces_all(pos, mass, N, G, delta, acc, nullptr, nthreads); ++nforce;                    // a(t+dt)
        for (int64_t k = 0; k < 3 * N; ++k) vel[k] = (vel[k] + vtilde[k]) / 2.0 + (dt / 2.0) * acc[k];  // (7)
    }
    return nforce;
}

// Half-kick / drift / half-kick form of the same scheme (reading R4).
int64_t oracle_kdk_halfkick(double* pos, double* vel, const double* mass, double* acc, int64_t N, double dt,
                            int64_t nsteps, double G, double delta, int acc_valid, int nthreads) {
    int64_t nforce = 0;
    if (!acc_valid) { forces_all(pos, mass, N, G, delta, acc, nullptr, nthreads); ++nforce; }
    for (int64_t s = 0; s < nsteps; ++s) {
        for (int64_t k = 0; k < 3 * N; ++k) vel[k] += (dt / 2.0) * acc[k];
        for (int64_t k = 0; k < 3 * N; ++k) pos[k] += dt * vel[k];
        forces_all(pos, mass, N, G, delta, acc, nullptr, nthreads); ++nforce;
        for (int64_t k = 0; k < 3 * N; ++k) vel[k] += (dt / 2.0) * acc[k];
    }
    return nforce;
}

// eqs. (8)-(10).  out16 = {E, K, W, Px, Py, Pz, Lx, Ly, Lz, Cx, Cy, Cz, M, 0, 0, 0}.
// pot (Phi_i, as returned by oracle_forces) may be NULL: it is then computed here.
void oracle_invariants(const double* pos, const double* vel, const double* mass, const double* pot, int64_t N,
                       double G, double delta, double* out16, int nthreads) {
    std::vector<double> phi;
    if (!pot) {
        phi.resize((size_t)N);
        std::vector<double> a((size_t)(3 * N));
        forces_all(pos, mass, N, G, delta, a.data(), phi.data(), nthreads);
        pot = phi.data();
    }
    NSum K, W, Px, Py, Pz, Lx, Ly, Lz, Cx, Cy, Cz, M;
    for (int64_t i = 0; i < N; ++i) {
        const double m = mass[i];
        const double x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
        const double u = vel[3 * i], v = vel[3 * i + 1], w = vel[3 * i + 2];
        K.add(0.5 * m * (u * u + v * v + w * w));       // first term of (8)
        W.add(0.5 * m * pot[i]);                         // second term of (8), sign and j != i per reading R3
        Px.add(m * u); Py.add(m * v); Pz.add(m * w);     // (9)
        Lx.add(m * (y * w - z * v));                     // (10) generalised to the full vector
        Ly.add(m * (z * u - x * w));
        Lz.add(m * (x * v - y * u));
        Cx.add(m * x); Cy.add(m * y); Cz.add(m * z);
        M.add(m);
    }
    const double Mt = M.value();
    out16[0] = K.value() + W.value();
    out16[1] = K.value();
    out16[2] = W.value();
    out16[3] = Px.value(); out16[4] = Py.value(); out16[5] = Pz.value();
    out16[6] = Lx.value(); out16[7] = Ly.value(); out16[8] = Lz.value();
    out16[9] = Cx.value() / Mt; out16[10] = Cy.value() / Mt; out16[11] = Cz.value() / Mt;
    out16[12] = Mt;
    out16[13] = out16[14] = out16[15] = 0.0;
}

int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
