// gg_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, double-precision CPU oracle for the explicit finite-volume step of the
// anisotropic, heterogeneous Gatenby-Gawlinski model (Mascia, Pera, Simeoni, arXiv 2006.01748).
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// call into this file.  It shares no source, header, table or helper with the CUDA path under
// paper_2006_01748_b200/csrc/ and neither side includes the other.
//
// What it computes -- the paper's scheme, written out literally:
//   eq. (3)     explicit Euler update of U, V, W, every right-hand side at time k;
//   Table 1  five-point stencil  D1(V;U)  for alpha * div((1-U) grad V);
//   Table 2  nine-point stencil  D2(W;A)  for div(A grad W), A=[[a,b],[b,c]];
//   Neumann boundaries: the paper prints no formula; reading A2 of
//   DESIGN.md is used: mirror (image) extension across every boundary face -- U,V,W,a,c even,
//   b odd -- which is the zero-normal-flux condition of the finite-volume scheme.
// The stencil entries are evaluated one by one in the tables' own form (weights times
// neighbour-minus-centre differences; centre weight = -(sum of the others), which equals the
// printed centre entries, see tests/test_oracle_pins.py).  No blocking, no fusion, no clamping.
//
// Index convention: arrays are row-major [ny][nx], i <-> x fastest, j <-> y; "right" = (i+1,j),
// "upper" = (i,j+1).  dx and dy are kept separate.
//
// Parity pins (tests/test_oracle_pins.py, -m "not gpu"): hand-computed 4x4 values for D1, D2 and
// one full step (tests/golden/*.txt), polynomial / plane-wave closed forms, uniform data -> ODE
// recursion, equilibria, conservation of sum W and sum V, 1-D reduction against an independent
// 1-D code, transpose / flip / rotation symmetries, discrete cosine eigenmodes over many steps,
// bounds for b = 0.  Nothing on this path is "parity unpinned".  (The NumPy reductions in
// oracle/__init__.py carry one unpinned item: the step-size RULE of max_stable_dt, reading A6.)
//
// Build: g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC (see oracle/build.py).  OpenMP only
// splits rows; every output cell depends on time-k data only, so the result is bit-identical for
// any thread count.

#include <cstddef>
#include <cstring>
#include <vector>

#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// O1: (ny+2) x (nx+2) copy of P with a one-cell ghost frame.  sign = +1: ghost = nearest
// interior cell (even mirror; corner ghosts = the corner cell, i.e. double mirror);
// sign = -1: ghost = minus the nearest interior cell (odd mirror, used for b only).
// [PAPER.md:42, :77 -- DESIGN.md reading A2, corner ghosts reading A12]
struct Padded {
    int nx, ny;
    std::vector<double> v;
    Padded(int nx_, int ny_) : nx(nx_), ny(ny_), v((size_t)(nx_ + 2) * (ny_ + 2)) {}
    // i in [-1, nx], j in [-1, ny]
    double& at(int i, int j) { return v[(size_t)(j + 1) * (nx + 2) + (i + 1)]; }
    double at(int i, int j) const { return v[(size_t)(j + 1) * (nx + 2) + (i + 1)]; }
    // nthreads only splits the row copies (pure data movement) over OpenMP threads.
    void fill(const double* P, double sign, int nthreads = 1) {
        (void)nthreads;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads)
#endif
        for (int j = 0; j < ny; ++j) {
            for (int i = 0; i < nx; ++i) at(i, j) = P[(size_t)j * nx + i];
            at(-1, j) = sign * at(0, j);
            at(nx, j) = sign * at(nx - 1, j);
        }
        for (int i = 0; i < nx; ++i) {
            at(i, -1) = sign * at(i, 0);
            at(i, ny) = sign * at(i, ny - 1);
        }
        // corner ghosts: mirror twice (sign * sign = +1 for both parities)
        at(-1, -1) = at(0, 0);
        at(nx, -1) = at(nx - 1, 0);
        at(-1, ny) = at(0, ny - 1);
        at(nx, ny) = at(nx - 1, ny - 1);
    }
};

// O3: D1(V;U)_ij, Table 1.
inline double D1_cell(const Padded& U, const Padded& V, int i, int j, double dx, double dy) {
    const double idx2 = 1.0 / (dx * dx), idy2 = 1.0 / (dy * dy);
    const double wE = idx2 - (U.at(i, j) + U.at(i + 1, j)) / (2.0 * dx * dx);
    const double wW = idx2 - (U.at(i - 1, j) + U.at(i, j)) / (2.0 * dx * dx);
    const double wN = idy2 - (U.at(i, j) + U.at(i, j + 1)) / (2.0 * dy * dy);
    const double wS = idy2 - (U.at(i, j - 1) + U.at(i, j)) / (2.0 * dy * dy);
    const double Vc = V.at(i, j);
    return wE * (V.at(i + 1, j) - Vc) + wW * (V.at(i - 1, j) - Vc) +
           wN * (V.at(i, j + 1) - Vc) + wS * (V.at(i, j - 1) - Vc);
}

// O5: D2(W;A)_ij, Table 2.  c here is the tensor entry c_T.
inline double D2_cell(const Padded& a, const Padded& b, const Padded& c, const Padded& W,
                      int i, int j, double dx, double dy) {
    const double E = (a.at(i, j) + a.at(i + 1, j)) / (2.0 * dx * dx);
    const double Wt = (a.at(i - 1, j) + a.at(i, j)) / (2.0 * dx * dx);
    const double N = (c.at(i, j) + c.at(i, j + 1)) / (2.0 * dy * dy);
    const double S = (c.at(i, j - 1) + c.at(i, j)) / (2.0 * dy * dy);
    const double NE = (b.at(i + 1, j) + b.at(i, j + 1)) / (4.0 * dx * dy);
    const double NW = -(b.at(i - 1, j) + b.at(i, j + 1)) / (4.0 * dx * dy);
    const double SE = -(b.at(i + 1, j) + b.at(i, j - 1)) / (4.0 * dx * dy);
    const double SW = (b.at(i - 1, j) + b.at(i, j - 1)) / (4.0 * dx * dy);
    const double Wc = W.at(i, j);
    return E * (W.at(i + 1, j) - Wc) + Wt * (W.at(i - 1, j) - Wc) +
           N * (W.at(i, j + 1) - Wc) + S * (W.at(i, j - 1) - Wc) +
           NE * (W.at(i + 1, j + 1) - Wc) + NW * (W.at(i - 1, j + 1) - Wc) +
           SE * (W.at(i + 1, j - 1) - Wc) + SW * (W.at(i - 1, j - 1) - Wc);
}

bool bad_shape(int nx, int ny, double dx, double dy) {
    return nx < 2 || ny < 2 || !(dx > 0.0) || !(dy > 0.0);
}

}  // namespace

extern "C" {

// D1(V;U) on the whole grid, Table 1.  out[ny][nx].
int gg_oracle_D1(int nx, int ny, double dx, double dy, const double* U, const double* V,
                 double* out) {
    if (bad_shape(nx, ny, dx, dy) || !U || !V || !out) return 1;
    Padded pU(nx, ny), pV(nx, ny);
    pU.fill(U, +1.0);
    pV.fill(V, +1.0);
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) out[(size_t)j * nx + i] = D1_cell(pU, pV, i, j, dx, dy);
    return 0;
}

// D2(W;A) on the whole grid, Table 2.  out[ny][nx].
int gg_oracle_D2(int nx, int ny, double dx, double dy, const double* a, const double* b,
                 const double* c, const double* W, double* out) {
    if (bad_shape(nx, ny, dx, dy) || !a || !b || !c || !W || !out) return 1;
    Padded pa(nx, ny), pb(nx, ny), pc(nx, ny), pW(nx, ny);
    pa.fill(a, +1.0);
    pb.fill(b, -1.0);
    pc.fill(c, +1.0);
    pW.fill(W, +1.0);
    for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i)
            out[(size_t)j * nx + i] = D2_cell(pa, pb, pc, pW, i, j, dx, dy);
    return 0;
}

// n explicit Euler steps of eq. (3) with constant step dt, in place on U, V, W ([ny][nx] each).
// c_r is the reaction parameter the paper calls c in eq. (1); (a, b, cT) is the tensor of eq. (2).
// nthreads <= 0: all OpenMP threads available.  Returns 0, or 1 on a bad argument.
int gg_oracle_step(int nx, int ny, double dx, double dy, double r, double d, double alpha,
                   double c_r, const double* a, const double* b, const double* cT, double* U,
                   double* V, double* W, long long n, double dt, int nthreads) {
    if (bad_shape(nx, ny, dx, dy) || !a || !b || !cT || !U || !V || !W || n < 0) return 1;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#else
    nthreads = 1;
#endif
    const size_t N = (size_t)nx * ny;
    Padded pa(nx, ny), pb(nx, ny), pc(nx, ny);
    pa.fill(a, +1.0);
    pb.fill(b, -1.0);
    pc.fill(cT, +1.0);
    Padded pU(nx, ny), pV(nx, ny), pW(nx, ny);
    std::vector<double> U1(N), V1(N), W1(N);
    for (long long k = 0; k < n; ++k) {
        // O1: ghost frames of the time-k fields
        pU.fill(U, +1.0, nthreads);
        pV.fill(V, +1.0, nthreads);
        pW.fill(W, +1.0, nthreads);
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads)
#endif
        for (int j = 0; j < ny; ++j) {
            for (int i = 0; i < nx; ++i) {
                const double u = pU.at(i, j), v = pV.at(i, j), w = pW.at(i, j);
                const size_t q = (size_t)j * nx + i;
                // O2: eq. (3) line 1
                U1[q] = u + dt * u * (1.0 - u) - d * dt * u * w;
                // O3 + O4: eq. (3) line 2
                V1[q] = v + r * dt * v * (1.0 - v) + alpha * dt * D1_cell(pU, pV, i, j, dx, dy);
                // O5 + O6: eq. (3) line 3
                W1[q] = w + c_r * dt * (v - w) + dt * D2_cell(pa, pb, pc, pW, i, j, dx, dy);
            }
        }
        // O7: swap; no clamping or positivity fix anywhere
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads)
#endif
        for (int j = 0; j < ny; ++j) {
            const size_t q = (size_t)j * nx, bytes = (size_t)nx * sizeof(double);
            std::memcpy(U + q, U1.data() + q, bytes);
            std::memcpy(V + q, V1.data() + q, bytes);
            std::memcpy(W + q, W1.data() + q, bytes);
        }
    }
    return 0;
}

int gg_oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
