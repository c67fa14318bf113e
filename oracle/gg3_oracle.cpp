// gg3_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, double-precision CPU oracle for the THREE-DIMENSIONAL extension of the explicit
// finite-volume step of the anisotropic, heterogeneous Gatenby-Gawlinski model (Mascia, Pera,
// Simeoni, arXiv 2006.01748).  Only tests/, __graft_entry__.smoke() and bench.py's reference legs
// may call into this file; it shares nothing with paper_2006_01748_b200/csrc/.
//
// The paper names the three-dimensional model only as the direction of its ongoing work
// and prints no 3-D scheme.  DESIGN.md reading A13 is used: the SAME construction
// as eq. (3) and Tables 1-2, one dimension up, on an nx x ny x nz Cartesian
// cell grid with spacings dx, dy, dz:
//
//   eq. (3)   explicit Euler, every right-hand side at time k, reactions unchanged;
//   Table 1'  seven-point stencil D1(V;U): one entry per face neighbour, weight
//             1/d^2 - (U_c + U_nb)/(2 d^2)  (d = the spacing across that face) -- Table 1's E, W,
//             N, S entries plus the same two along z; centre = -(sum of the six);
//   Table 2'  nineteen-point stencil D2(W;A) for div(A grad W) with the symmetric tensor
//             A = [[axx,axy,axz],[axy,ayy,ayz],[axz,ayz,azz]]: six face entries
//             (a_c + a_nb)/(2 d^2) with the diagonal entry of that direction -- Table 2's E, W, N, S
//             -- and, for EACH of the three coordinate planes, Table 2's four corner entries with
//             that plane's off-diagonal entry:  +-(a_pq at the p-neighbour + a_pq at the
//             q-neighbour)/(4 dp dq), sign + for the (+,+) and (-,-) corners, - for the mixed ones
//             (nested central differences dp(a_pq dq W) + dq(a_pq dp W)); centre = -(sum of the 18).
//   Neumann boundaries: the mirror extension of reading A2 -- U, V, W and the diagonal entries
//   even across every boundary face; an off-diagonal entry a_pq odd across the faces normal to p
//   or q, even across the faces normal to the third axis (a reflection R maps A to R A R).
//
// Stencil entries are evaluated one by one as weight x (neighbour - centre).  The four in-plane
// terms of Table 2 come first and in D2_cell's order, then the z faces, then the xz and yz
// corners, so that z-uniform data with axz = ayz = 0 reproduces the 2-D oracle bit for bit.
//
// Index convention: arrays are [nz][ny][nx], i <-> x fastest, then j <-> y, then k <-> z.
//
// Parity pins (tests/test_oracle3d_pins.py, -m "not gpu"): nested-central-difference brute force
// in pure Python on tiny grids; polynomial closed forms for each tensor entry (sign and factor of
// every cross term); the plane-wave symbol; z-, y- and x-uniform data against the pinned 2-D oracle
// (bit for bit for z); axis permutations; sum W and sum V conserved with all three off-diagonals
// non-zero; uniform data == scalar recursion; equilibria.  The SCHEME is reading A13 (the paper
// prints none): "parity unpinned" as far as the choice of scheme goes, pinned against the
// mathematics it states.
//
// Build: with gg_oracle.cpp into oracle/libgg_oracle.so (oracle/build.py), same flags.

#include <cstddef>
#include <cstring>
#include <vector>

#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// (nz+2) x (ny+2) x (nx+2) copy of P with a one-cell ghost frame.  sx, sy, sz = +1 / -1: parity of
// the field under reflection across the faces normal to x, y, z; ghosts on edges and corners are
// mirrored once per axis they stick out along (signs multiply).
struct Padded3 {
    int nx, ny, nz;
    std::vector<double> v;
    Padded3(int nx_, int ny_, int nz_) : nx(nx_), ny(ny_), nz(nz_), v((size_t)(nx_ + 2) * (ny_ + 2) * (nz_ + 2)) {}
    double& at(int i, int j, int k) { return v[((size_t)(k + 1) * (ny + 2) + (j + 1)) * (nx + 2) + (i + 1)]; }
    double at(int i, int j, int k) const { return v[((size_t)(k + 1) * (ny + 2) + (j + 1)) * (nx + 2) + (i + 1)]; }
    void fill(const double* P, double sx, double sy, double sz) {
        for (int k = -1; k <= nz; ++k) {
            const int kk = k < 0 ? 0 : k >= nz ? nz - 1 : k;
            const double fz = (k < 0 || k >= nz) ? sz : 1.0;
            for (int j = -1; j <= ny; ++j) {
                const int jj = j < 0 ? 0 : j >= ny ? ny - 1 : j;
                const double fy = (j < 0 || j >= ny) ? sy : 1.0;
                for (int i = -1; i <= nx; ++i) {
                    const int ii = i < 0 ? 0 : i >= nx ? nx - 1 : i;
                    const double fx = (i < 0 || i >= nx) ? sx : 1.0;
                    at(i, j, k) = fx * fy * fz * P[((size_t)kk * ny + jj) * nx + ii];
                }
            }
        }
    }
};

// Table 1', one entry per face neighbour.
inline double D1_cell3(const Padded3& U, const Padded3& V, int i, int j, int k, double dx, double dy, double dz) {
    const double idx2 = 1.0 / (dx * dx), idy2 = 1.0 / (dy * dy), idz2 = 1.0 / (dz * dz);
    const double Uc = U.at(i, j, k), Vc = V.at(i, j, k);
    const double wE = idx2 - (Uc + U.at(i + 1, j, k)) / (2.0 * dx * dx);
    const double wW = idx2 - (U.at(i - 1, j, k) + Uc) / (2.0 * dx * dx);
    const double wN = idy2 - (Uc + U.at(i, j + 1, k)) / (2.0 * dy * dy);
    const double wS = idy2 - (U.at(i, j - 1, k) + Uc) / (2.0 * dy * dy);
    const double wT = idz2 - (Uc + U.at(i, j, k + 1)) / (2.0 * dz * dz);
    const double wB = idz2 - (U.at(i, j, k - 1) + Uc) / (2.0 * dz * dz);
    return wE * (V.at(i + 1, j, k) - Vc) + wW * (V.at(i - 1, j, k) - Vc) +
           wN * (V.at(i, j + 1, k) - Vc) + wS * (V.at(i, j - 1, k) - Vc) +
           wT * (V.at(i, j, k + 1) - Vc) + wB * (V.at(i, j, k - 1) - Vc);
}

struct Tensor3 {
    Padded3 xx, yy, zz, xy, xz, yz;
    Tensor3(int nx, int ny, int nz) : xx(nx, ny, nz), yy(nx, ny, nz), zz(nx, ny, nz), xy(nx, ny, nz), xz(nx, ny, nz), yz(nx, ny, nz) {}
    void fill(const double* axx, const double* ayy, const double* azz, const double* axy, const double* axz, const double* ayz) {
        xx.fill(axx, +1, +1, +1);
        yy.fill(ayy, +1, +1, +1);
        zz.fill(azz, +1, +1, +1);
        xy.fill(axy, -1, -1, +1);
        xz.fill(axz, -1, +1, -1);
        yz.fill(ayz, +1, -1, -1);
    }
};

// Table 2', entry by entry.
inline double D2_cell3(const Tensor3& A, const Padded3& W, int i, int j, int k, double dx, double dy, double dz) {
    const double Wc = W.at(i, j, k);
    // the xy plane: Table 2 as printed, a = axx, b = axy, c = ayy
    const double E = (A.xx.at(i, j, k) + A.xx.at(i + 1, j, k)) / (2.0 * dx * dx);
    const double Wt = (A.xx.at(i - 1, j, k) + A.xx.at(i, j, k)) / (2.0 * dx * dx);
    const double N = (A.yy.at(i, j, k) + A.yy.at(i, j + 1, k)) / (2.0 * dy * dy);
    const double S = (A.yy.at(i, j - 1, k) + A.yy.at(i, j, k)) / (2.0 * dy * dy);
    const double NE = (A.xy.at(i + 1, j, k) + A.xy.at(i, j + 1, k)) / (4.0 * dx * dy);
    const double NW = -(A.xy.at(i - 1, j, k) + A.xy.at(i, j + 1, k)) / (4.0 * dx * dy);
    const double SE = -(A.xy.at(i + 1, j, k) + A.xy.at(i, j - 1, k)) / (4.0 * dx * dy);
    const double SW = (A.xy.at(i - 1, j, k) + A.xy.at(i, j - 1, k)) / (4.0 * dx * dy);
    double s = E * (W.at(i + 1, j, k) - Wc) + Wt * (W.at(i - 1, j, k) - Wc) +
               N * (W.at(i, j + 1, k) - Wc) + S * (W.at(i, j - 1, k) - Wc) +
               NE * (W.at(i + 1, j + 1, k) - Wc) + NW * (W.at(i - 1, j + 1, k) - Wc) +
               SE * (W.at(i + 1, j - 1, k) - Wc) + SW * (W.at(i - 1, j - 1, k) - Wc);
    // the z faces
    const double T = (A.zz.at(i, j, k) + A.zz.at(i, j, k + 1)) / (2.0 * dz * dz);
    const double B = (A.zz.at(i, j, k - 1) + A.zz.at(i, j, k)) / (2.0 * dz * dz);
    s += T * (W.at(i, j, k + 1) - Wc) + B * (W.at(i, j, k - 1) - Wc);
    // the xz plane: the same four corner entries with axz
    const double TE = (A.xz.at(i + 1, j, k) + A.xz.at(i, j, k + 1)) / (4.0 * dx * dz);
    const double TW = -(A.xz.at(i - 1, j, k) + A.xz.at(i, j, k + 1)) / (4.0 * dx * dz);
    const double BE = -(A.xz.at(i + 1, j, k) + A.xz.at(i, j, k - 1)) / (4.0 * dx * dz);
    const double BW = (A.xz.at(i - 1, j, k) + A.xz.at(i, j, k - 1)) / (4.0 * dx * dz);
    s += TE * (W.at(i + 1, j, k + 1) - Wc) + TW * (W.at(i - 1, j, k + 1) - Wc) +
         BE * (W.at(i + 1, j, k - 1) - Wc) + BW * (W.at(i - 1, j, k - 1) - Wc);
    // the yz plane, with ayz
    const double TN = (A.yz.at(i, j + 1, k) + A.yz.at(i, j, k + 1)) / (4.0 * dy * dz);
    const double TS = -(A.yz.at(i, j - 1, k) + A.yz.at(i, j, k + 1)) / (4.0 * dy * dz);
    const double BN = -(A.yz.at(i, j + 1, k) + A.yz.at(i, j, k - 1)) / (4.0 * dy * dz);
    const double BS = (A.yz.at(i, j - 1, k) + A.yz.at(i, j, k - 1)) / (4.0 * dy * dz);
    s += TN * (W.at(i, j + 1, k + 1) - Wc) + TS * (W.at(i, j - 1, k + 1) - Wc) +
         BN * (W.at(i, j + 1, k - 1) - Wc) + BS * (W.at(i, j - 1, k - 1) - Wc);
    return s;
}

bool bad_shape3(int nx, int ny, int nz, double dx, double dy, double dz) {
    return nx < 2 || ny < 2 || nz < 2 || !(dx > 0.0) || !(dy > 0.0) || !(dz > 0.0);
}

}  // namespace

extern "C" {

int gg3_oracle_D1(int nx, int ny, int nz, double dx, double dy, double dz, const double* U, const double* V, double* out) {
    if (bad_shape3(nx, ny, nz, dx, dy, dz) || !U || !V || !out) return 1;
    Padded3 pU(nx, ny, nz), pV(nx, ny, nz);
    pU.fill(U, +1, +1, +1);
    pV.fill(V, +1, +1, +1);
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) out[((size_t)k * ny + j) * nx + i] = D1_cell3(pU, pV, i, j, k, dx, dy, dz);
    return 0;
}

// tensor: six arrays in the order axx, ayy, azz, axy, axz, ayz
int gg3_oracle_D2(int nx, int ny, int nz, double dx, double dy, double dz, const double* axx, const double* ayy,
                  const double* azz, const double* axy, const double* axz, const double* ayz, const double* W, double* out) {
    if (bad_shape3(nx, ny, nz, dx, dy, dz) || !axx || !ayy || !azz || !axy || !axz || !ayz || !W || !out) return 1;
    Tensor3 A(nx, ny, nz);
    A.fill(axx, ayy, azz, axy, axz, ayz);
    Padded3 pW(nx, ny, nz);
    pW.fill(W, +1, +1, +1);
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) out[((size_t)k * ny + j) * nx + i] = D2_cell3(A, pW, i, j, k, dx, dy, dz);
    return 0;
}

// n explicit Euler steps of eq. (3) in three dimensions, in place on U, V, W ([nz][ny][nx] each).
int gg3_oracle_step(int nx, int ny, int nz, double dx, double dy, double dz, double r, double d, double alpha, double c_r,
                    const double* axx, const double* ayy, const double* azz, const double* axy, const double* axz,
                    const double* ayz, double* U, double* V, double* W, long long n, double dt, int nthreads) {
    if (bad_shape3(nx, ny, nz, dx, dy, dz) || !axx || !ayy || !azz || !axy || !axz || !ayz || !U || !V || !W || n < 0) return 1;
#ifdef _OPENMP
    if (nthreads <= 0) nthreads = omp_get_max_threads();
#else
    nthreads = 1;
#endif
    const size_t N = (size_t)nx * ny * nz;
    Tensor3 A(nx, ny, nz);
    A.fill(axx, ayy, azz, axy, axz, ayz);
    Padded3 pU(nx, ny, nz), pV(nx, ny, nz), pW(nx, ny, nz);
    std::vector<double> U1(N), V1(N), W1(N);
    for (long long s = 0; s < n; ++s) {
        pU.fill(U, +1, +1, +1);
        pV.fill(V, +1, +1, +1);
        pW.fill(W, +1, +1, +1);
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(nthreads)
#endif
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    const double u = pU.at(i, j, k), v = pV.at(i, j, k), w = pW.at(i, j, k);
                    const size_t q = ((size_t)k * ny + j) * nx + i;
                    U1[q] = u + dt * u * (1.0 - u) - d * dt * u * w;
                    V1[q] = v + r * dt * v * (1.0 - v) + alpha * dt * D1_cell3(pU, pV, i, j, k, dx, dy, dz);
                    W1[q] = w + c_r * dt * (v - w) + dt * D2_cell3(A, pW, i, j, k, dx, dy, dz);
                }
        std::memcpy(U, U1.data(), N * sizeof(double));
        std::memcpy(V, V1.data(), N * sizeof(double));
        std::memcpy(W, W1.data(), N * sizeof(double));
    }
    return 0;
}

}  // extern "C"
