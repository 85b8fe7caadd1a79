/* tdse_oracle.c -- serial CPU oracle for the FDTD hot path of arXiv 2401.07416.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call this.  It shares no code,
 * header, table or helper with paper_2401_07416_b200/ (the CUDA path); neither imports
 * the other.  Plain C, one cell at a time, in the paper's order and notation, so it can
 * be checked against PAPER.md by eye.  Build: gcc -O2 -ffp-contract=off [-fopenmp].
 * The optional OpenMP pragma parallelises the k loop of one half-step only; every cell
 * is independent within a half-step, so results are bit-identical to the serial run.
 *
 * What each function follows:
 *   oracle_potential   BASELINE.json north_star (1) + configs: V = clamp( sum_a -Z_a exp(-r_a/lambda_a)
 *                      / sqrt(r_a^2 + s_a^2) ); nearest image on periodic axes (reading 15).
 *                      Stands in for the DFT potential of PAPER.md:50, 164.
 *   oracle_mask        absorbing layer, PAPER.md:89-94 (eq 10) read as a polynomial mask
 *                      (reading 6).
 *   oracle_wavepacket  eq (3), with a signed wave vector (readings 2, 3, 5).
 *   oracle_stagger     I^{-1/2} = Im psi0 + (1/2) A Re psi0   (reading 4).
 *   oracle_step_*      eqs (8), (9), (13), (14), (15): see tdse_oracle_step.inc.
 *   oracle_norm_*      PAPER.md:87 density and the conserved Visscher form.
 *   oracle_plane_density_*  one detector frame rho(i,j) = R^2 + I^2 on plane k_det (eq (15)).
 *   oracle_potential_cell   unit-cell potential tiled in x, y and interpolated onto the mesh (
 *                           DESIGN.md reading 24).
 *   oracle_dissimilarity    eq (16), between two frame trajectories (reading 23).
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): dense-eigh closed form on tiny grids, FFT
 * closed form, exact expm propagation + second-order convergence, conservation of q_visscher,
 * stationary eigenvector, harmonic-oscillator ground state, free Gaussian closed form,
 * blow-up past the stability bound, analytic single-atom potential, mask invariants,
 * detector identities.  Parity unpinned: nothing paper-specific (its Cu/Au DFT potentials,
 * its 879 trajectories) -- that data is not available.
 */
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

enum { BC_PERIODIC = 0, BC_DIRICHLET = 1 };

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* V(i,j,k) = clamp( sum_a -Z_a * screen_a(r_a) / sqrt(r_a^2 + s_a^2), vmin, vmax )
 * atoms: natoms records (x, y, z, Z, s^2, lambda); lambda <= 0 or non-finite: screen = 1.
 * r_a: distance from the grid point (i dx, j dy, k dz) to the atom; on a
 * periodic axis the displacement is reduced to the nearest image, d <- d - L round(d/L).
 * rcut > 0: atoms with r_a > rcut are skipped.  Sum in list order, double throughout. */
void oracle_potential(int nx, int ny, int nz, double dx, double dy, double dz, int bcx, int bcy, int bcz,
                      const double* atoms, int natoms, double vmin, double vmax, double rcut,
                      double* V)
{
    const double Lx = nx * dx, Ly = ny * dy, Lz = nz * dz;
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                const double x = i * dx, y = j * dy, z = k * dz;
                double sum = 0.0;
                for (int a = 0; a < natoms; ++a) {
                    const double* A = atoms + 6 * (size_t)a;
                    double ddx = x - A[0], ddy = y - A[1], ddz = z - A[2];
                    if (bcx == BC_PERIODIC) ddx = ddx - Lx * round(ddx / Lx);
                    if (bcy == BC_PERIODIC) ddy = ddy - Ly * round(ddy / Ly);
                    if (bcz == BC_PERIODIC) ddz = ddz - Lz * round(ddz / Lz);
                    const double r2 = ddx * ddx + ddy * ddy + ddz * ddz;
                    const double r = sqrt(r2);
                    if (rcut > 0.0 && r > rcut) continue;
                    double screen = 1.0;
                    if (A[5] > 0.0 && isfinite(A[5])) screen = exp(-r / A[5]);
                    sum += -A[3] * screen / sqrt(r2 + A[4]);
                }
                if (sum < vmin) sum = vmin;
                if (sum > vmax) sum = vmax;
                V[((size_t)k * ny + j) * nx + i] = sum;
            }
}

/* M[k] = 1 - strength * xi_k^power, xi = (w_lo - k)/w_lo for k < w_lo (low-z layer),
 * xi = (k - (nz-1-w_hi))/w_hi for k > nz-1-w_hi (high-z layer), M = 1 elsewhere. */
void oracle_mask(int nz, int w_lo, int w_hi, double strength, int power, double* M)
{
    for (int k = 0; k < nz; ++k) {
        double xi = 0.0;
        if (w_lo > 0 && k < w_lo) xi = (double)(w_lo - k) / (double)w_lo;
        if (w_hi > 0 && k > nz - 1 - w_hi) xi = (double)(k - (nz - 1 - w_hi)) / (double)w_hi;
        double p = 1.0;
        for (int q = 0; q < power; ++q) p *= xi;
        M[k] = (xi > 0.0) ? 1.0 - strength * p : 1.0;
    }
}

/* psi0 = N exp(-|r - r0|^2 / (2 sigma^2)) exp(+i k0.(r - r0)), eq (3) with the paper's
 * case k0 = (0, 0, -2 pi / lambda).  amplitude == 0: N = (pi sigma^2)^(-3/4).
 * Outputs R0 = Re psi0, J0 = Im psi0 (double). */
void oracle_wavepacket(int nx, int ny, int nz, double dx, double dy, double dz,
                       double x0, double y0, double z0, double sigma,
                       double kx, double ky, double kz, double amplitude,
                       double* R0, double* J0)
{
    const double pi = 3.14159265358979323846;
    const double N = (amplitude != 0.0) ? amplitude : pow(pi * sigma * sigma, -0.75);
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                const double ddx = i * dx - x0, ddy = j * dy - y0, ddz = k * dz - z0;
                const double G = N * exp(-(ddx * ddx + ddy * ddy + ddz * ddz) / (2.0 * sigma * sigma));
                const double phi = kx * ddx + ky * ddy + kz * ddz;
                const size_t p = ((size_t)k * ny + j) * nx + i;
                R0[p] = G * cos(phi);
                J0[p] = G * sin(phi);
            }
}

static inline double at_d(const double* f, int nx, int ny, int nz, int bcx, int bcy, int bcz,
                          int i, int j, int k)
{
    if (i < 0)   { if (bcx == BC_PERIODIC) i = nx - 1; else return 0.0; }
    if (i >= nx) { if (bcx == BC_PERIODIC) i = 0;      else return 0.0; }
    if (j < 0)   { if (bcy == BC_PERIODIC) j = ny - 1; else return 0.0; }
    if (j >= ny) { if (bcy == BC_PERIODIC) j = 0;      else return 0.0; }
    if (k < 0)   { if (bcz == BC_PERIODIC) k = nz - 1; else return 0.0; }
    if (k >= nz) { if (bcz == BC_PERIODIC) k = 0;      else return 0.0; }
    return f[((size_t)k * ny + j) * nx + i];
}

/* I^{-1/2} = J0 + (1/2) (A R0),  (A f) = -c_x d2x f - c_y d2y f - c_z d2z f + c_v V f
 * (A = dt H / hbar, H from eq (2)).  V is the potential as stored (already rounded
 * to the run's dtype, passed here as double); R0, J0 unrounded doubles. */
void oracle_stagger(int nx, int ny, int nz, int bcx, int bcy, int bcz,
                    double cx, double cy, double cz, double cv,
                    const double* V, const double* R0, const double* J0, double* Ihalf)
{
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                const size_t p = ((size_t)k * ny + j) * nx + i;
                const double r = R0[p];
                const double d2x = at_d(R0, nx, ny, nz, bcx, bcy, bcz, i + 1, j, k) - 2.0 * r
                                 + at_d(R0, nx, ny, nz, bcx, bcy, bcz, i - 1, j, k);
                const double d2y = at_d(R0, nx, ny, nz, bcx, bcy, bcz, i, j + 1, k) - 2.0 * r
                                 + at_d(R0, nx, ny, nz, bcx, bcy, bcz, i, j - 1, k);
                const double d2z = at_d(R0, nx, ny, nz, bcx, bcy, bcz, i, j, k + 1) - 2.0 * r
                                 + at_d(R0, nx, ny, nz, bcx, bcy, bcz, i, j, k - 1);
                const double Ar = -cx * d2x - cy * d2y - cz * d2z + cv * V[p] * r;
                Ihalf[p] = J0[p] + 0.5 * Ar;
            }
}

#define REAL double
#define NAME(x) x##_f64
#include "tdse_oracle_step.inc"
#undef REAL
#undef NAME

#define REAL float
#define NAME(x) x##_f32
#include "tdse_oracle_step.inc"
#undef REAL
#undef NAME

/* Dissimilarity of two detector-plane trajectories, eq (16) PAPER.md:219-221:
 *   d_kj = 1/(t1 - t0) * int_{t0}^{t1} ( int_D ( rho_k(r,t) - rho_j(r,t) )^2 dr )^{1/2} dt
 * rho_k, rho_j: [nframes][npix] frames of |psi|^2 on the detector plane at equally spaced times.
 * Reading: int_D dr -> dA * sum over pixels; the time average over the window
 * [t0, t1] -> the arithmetic mean over the frames s0 .. s1 (inclusive) that fall in it.
 * Serial sums in double, pixels in row-major order, frames in increasing order. */
double oracle_dissimilarity(const double* rho_k, const double* rho_j, int npix, double dA, int s0, int s1)
{
    double acc = 0.0;
    for (int s = s0; s <= s1; ++s) {
        double inner = 0.0;
        for (int p = 0; p < npix; ++p) {
            const double d = rho_k[(size_t)s * npix + p] - rho_j[(size_t)s * npix + p];
            inner += d * d;
        }
        acc += sqrt(dA * inner);
    }
    return acc / (double)(s1 - s0 + 1);
}

/* Potential from a unit-cell grid ("the values of the electrostatic potential at each grid point
 * V(i,j,k) were obtained by interpolating the calculated potential"; PAPER.md:213 step (ii) "expansion and
 * interpolation of the electrostatic potential onto the mesh points").  Reading: the unit cell
 * holds cell[mz][my][mx] samples at spacings (ax/mx, ay/my, az/(mz-1)); it repeats periodically in x and y (the
 * slab's supercell expansion) and is sampled by trilinear interpolation at the mesh point
 * (i dx - x0, j dy - y0, k dz - z0); below z0 and above z0 + az the nearest z plane is used.  Then clamp. */
void oracle_potential_cell(int nx, int ny, int nz, double dx, double dy, double dz,
                           const double* cell, int mx, int my, int mz, double ax, double ay, double az,
                           double x0, double y0, double z0, double vmin, double vmax, double* V)
{
    const double hx = ax / mx, hy = ay / my, hz = (mz > 1) ? az / (mz - 1) : 1.0;
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                double u = (i * dx - x0) / hx, v = (j * dy - y0) / hy, w = (k * dz - z0) / hz;
                if (w < 0.0) w = 0.0;
                if (w > (double)(mz - 1)) w = (double)(mz - 1);
                const double fu = floor(u), fv = floor(v), fw = floor(w);
                const double tu = u - fu, tv = v - fv;
                int iw0 = (int)fw;
                if (iw0 > mz - 2) iw0 = (mz > 1) ? mz - 2 : 0;
                const double tw = (mz > 1) ? w - (double)iw0 : 0.0;
                const int iw1 = (mz > 1) ? iw0 + 1 : 0;
                long long iu0 = (long long)fu % mx; if (iu0 < 0) iu0 += mx;
                long long iv0 = (long long)fv % my; if (iv0 < 0) iv0 += my;
                const long long iu1 = (iu0 + 1) % mx, iv1 = (iv0 + 1) % my;
#define CELL(a, b, c) cell[((size_t)(c) * my + (size_t)(b)) * mx + (size_t)(a)]
                const double c00 = CELL(iu0, iv0, iw0) * (1.0 - tu) + CELL(iu1, iv0, iw0) * tu;
                const double c10 = CELL(iu0, iv1, iw0) * (1.0 - tu) + CELL(iu1, iv1, iw0) * tu;
                const double c01 = CELL(iu0, iv0, iw1) * (1.0 - tu) + CELL(iu1, iv0, iw1) * tu;
                const double c11 = CELL(iu0, iv1, iw1) * (1.0 - tu) + CELL(iu1, iv1, iw1) * tu;
#undef CELL
                const double c0 = c00 * (1.0 - tv) + c10 * tv;
                const double c1 = c01 * (1.0 - tv) + c11 * tv;
                double val = c0 * (1.0 - tw) + c1 * tw;
                if (val < vmin) val = vmin;
                if (val > vmax) val = vmax;
                V[((size_t)k * ny + j) * nx + i] = val;
            }
}
