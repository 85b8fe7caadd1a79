// tdse_kernels_basic.cuh -- set-up kernels (potential, packet, raw fills), the two-pass
// reference stencil (one thread per cell), detector and norm reductions.
// Citations: PAPER.md = /root/reference/PAPER.md (arXiv 2401.07416).
#pragma once
#include "tdse_common.cuh"

namespace tdse {

struct AtomRec { double x, y, z, Z, soft2, screen; };   // same layout as tdse_atom

// ---------------------------------------------------------------------------------------------
// S0 potential build (BASELINE.json north_star (1)): V = clamp(sum_a -Z_a exp(-r_a/lambda_a)/sqrt(r_a^2+s_a^2)).
// Bound by the fp64 pipe, so the work per cell-atom pair is cut down to ~35 fp64 instructions without branches:
//   * a thread owns CELLS consecutive cells along x and shares the y/z part of the distance among them;
//   * atoms are staged through shared memory in chunks with 1/lambda precomputed;
//   * r and 1/sqrt(r^2+s^2): the hardware seed (MUFU.RSQ64H through rsqrt.approx.ftz.f64) + one third-order step each;
//   * exp(-r/lambda): x = n ln2/256 + r, exp(x) = 2^(n div 256) * T[n mod 256] * (1 + q(r)), T[j] = 2^(j/256) in shared
//     memory, q = expm1 as a degree-4 polynomial on |r| <= ln2/512 (remainder < 4e-17);
//   * nearest image by the round-to-nearest-even magic constant instead of rint.
// Double accumulate in list order, one rounding to `real`.  One launch covers every batch entry (blockIdx.y); the
// sum may start from a per-cell prefix (the atoms all entries share, summed once: prefix_out mode) -- the same sequence of
// fma as the plain list-order sum, so the result does not depend on whether the prefix was shared.
// ---------------------------------------------------------------------------------------------
constexpr int kAtomChunk = 128;

struct AtomStaged { double x, y, z, Z, soft2, inv_screen; };   // inv_screen = 0: unscreened
struct AtomRange { int first, count; };                        // one entry's slice of the atom array

constexpr double kRoundMagic = 6755399441055744.0;             // 1.5 * 2^52: x + magic - magic = x rounded to nearest even

// 1/sqrt(a) for normal a > 0: ~22-bit hardware seed, then y (1 + e/2 + 3 e^2/8) with e = 1 - a y^2 (error O(e^3))
__device__ __forceinline__ double rsqrt_pos(double a)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    const double t = a * y;
    const double e = fma(-t, y, 1.0);
    const double p = fma(0.375, e, 0.5);
    return fma(y * e, p, y);
}

// sqrt(a) for normal a > 0 from the same seed: a y is already sqrt(a) to 22 bits, and sqrt(a) = a y (1 + e/2 + 3 e^2/8)
__device__ __forceinline__ double sqrt_pos(double a)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    const double t = a * y;
    const double e = fma(-t, y, 1.0);
    const double p = fma(0.375, e, 0.5);
    return fma(t * e, p, t);
}

// exp(x) for -30000 < x <= 0 with the 2^(j/256) table `T` (shared memory): x = n ln2/256 + r, |r| <= ln2/512, and
// exp(x) = 2^(n div 256) * T[n mod 256] * (1 + q(r)), q = expm1 as a degree-4 polynomial (remainder r^5/120 < 4e-17).
// r comes from one fma with ln2/256 rounded to double: its error, |n| * 2^-61, stays below 2e-15 for every term that
// is not itself below 1e-16 (|x| < 37).  Below x = -708 the result stays near 2^-1022, which no sum registers.  exp(-0) = 1.
// x is clamped at -746 first (one DMNMX): a screening length far below the mesh (or a denormal one, inv_screen = inf)
// gives x = -1e10 or -inf, where the integer n would wrap and r = inf - inf; the clamp turns those into "about 2^-1022",
// which is what exp underflows to.  Every x > -746 goes through unchanged.
constexpr int kExpTable = 256;

__device__ __forceinline__ double exp_nonpositive(double x, const double* __restrict__ T)
{
    x = fmax(x, -746.0);
    double t = fma(x, (double)kExpTable * 1.4426950408889634074, kRoundMagic);
    const int n = max(__double2loint(t), -1022 * kExpTable);        // n = 256 k + j; k >= -1022 keeps the result a normal number
    t -= kRoundMagic;
    const double r = fma(t, -0.69314718055994530942 / (double)kExpTable, x);
    double p = fma(r, 1.0 / 24.0, 1.0 / 6.0);
    p = fma(p, r, 0.5);
    p = fma(p, r, 1.0);
    const double s = T[n & (kExpTable - 1)];
    const double v = fma(s, p * r, s);                              // 2^(j/256) e^r in [0.5, 2)
    return __hiloint2double(__double2hiint(v) + ((n >> 8) << 20), __double2loint(v));   // * 2^k
}

// distance from coordinate a to the interval [lo, hi] along one axis (nearest periodic image if L > 0)
__device__ __forceinline__ double axis_gap(double a, double lo, double hi, double L)
{
    if (L > 0.0) a -= L * floor(a / L);   // the pair test takes any number of periods: bring a into [0, L) first
    double g = fmax(0.0, fmax(lo - a, a - hi));
    if (L > 0.0) {
        g = fmin(g, fmax(0.0, fmax(lo - (a + L), (a + L) - hi)));
        g = fmin(g, fmax(0.0, fmax(lo - (a - L), (a - L) - hi)));
    }
    return g;
}

// A block owns a brick of kPotBX x kPotBY x kPotBZ threads = (CELLS kPotBX) x kPotBY x kPotBZ cells of entry blockIdx.y.
// HAS_CUT: atoms farther than rcut from every cell of the brick are dropped while the list is staged (ordered
// compaction, so the summation order of the kept atoms is the list order); the pair test itself is that of the definition (include/tdse.h).
// PREFIX_OUT: write the unclamped fp64 sums to `prefix_out` (flat [nz][ny][nx]) instead of V.
constexpr int kPotBX = 16, kPotBY = 4, kPotBZ = 4;

template <typename real, int CELLS, bool HAS_CUT, bool PREFIX_OUT>
__global__ void __launch_bounds__(256, 3)
potential_build_kernel(Grid g, double dx, double dy, double dz, const AtomRec* __restrict__ atoms,
                       const AtomRange* __restrict__ ranges /* [gridDim.y] or NULL */, int first0, int count0,
                       const double* __restrict__ prefix_in /* flat fp64 sums of the atoms before `first`, or NULL */,
                       double vmin, double vmax, double rcut, real* __restrict__ V /* base of entry blockIdx.y = 0 */,
                       double* __restrict__ prefix_out)
{
    static_assert(kPotBX * kPotBY * kPotBZ == 256 && kAtomChunk <= 256, "block shape");
    __shared__ AtomStaged s_atoms[kAtomChunk];
    __shared__ double s_exp2[kExpTable];
    __shared__ int s_warp_count[8];
    const int tx = threadIdx.x % kPotBX, ty = (threadIdx.x / kPotBX) % kPotBY, tz = threadIdx.x / (kPotBX * kPotBY);
    const int bricks_x = (g.nx + CELLS * kPotBX - 1) / (CELLS * kPotBX), bricks_y = (g.ny + kPotBY - 1) / kPotBY;
    const int bx = blockIdx.x % bricks_x, by = (blockIdx.x / bricks_x) % bricks_y, bz = blockIdx.x / (bricks_x * bricks_y);
    const int i0 = (bx * kPotBX + tx) * CELLS, j = by * kPotBY + ty, k = bz * kPotBZ + tz;
    const bool live = i0 < g.nx && j < g.ny && k < g.nz;
    const int first = ranges ? ranges[blockIdx.y].first : first0;
    const int natoms = ranges ? ranges[blockIdx.y].count : count0;
    const double y = j * dy, z = k * dz;
    const double Lx = g.nx * dx, Ly = g.ny * dy, Lz = g.nz * dz;
    const double iLx = 1.0 / Lx, iLy = 1.0 / Ly, iLz = 1.0 / Lz;
    const bool perx = g.bcx == BC_PERIODIC, pery = g.bcy == BC_PERIODIC, perz = g.bcz == BC_PERIODIC;
    const double rc2 = rcut * rcut;
    // the brick's bounding box, padded by a cell so that rounding never drops an atom the pair test would keep
    const double lox = (bx * kPotBX * CELLS - 1) * dx, hix = ((bx + 1) * kPotBX * CELLS) * dx;
    const double loy = (by * kPotBY - 1) * dy, hiy = ((by + 1) * kPotBY) * dy;
    const double loz = (bz * kPotBZ - 1) * dz, hiz = ((bz + 1) * kPotBZ) * dz;
    static_assert(kExpTable == 256, "n >> 8 above");
    if (threadIdx.x < kExpTable) s_exp2[threadIdx.x] = exp2((double)threadIdx.x / (double)kExpTable);
    double sum[CELLS], xs[CELLS];
#pragma unroll
    for (int e = 0; e < CELLS; ++e) xs[e] = (i0 + e) * dx;
    const long long flat0 = ((long long)k * g.ny + j) * g.nx + i0;
#pragma unroll
    for (int e = 0; e < CELLS; ++e) sum[e] = (prefix_in && live && i0 + e < g.nx) ? prefix_in[flat0 + e] : 0.0;
    for (int a0 = 0; a0 < natoms; a0 += kAtomChunk) {
        const int nc = min(kAtomChunk, natoms - a0);
        __syncthreads();                                  // previous chunk fully consumed (first pass: table written)
        // ---- stage: thread q < nc looks at atom first + a0 + q ----
        int na = nc;
        {
            AtomStaged S;
            bool keep = false;
            if (threadIdx.x < nc) {
                const AtomRec A = atoms[first + a0 + threadIdx.x];
                S.x = A.x; S.y = A.y; S.z = A.z; S.Z = A.Z; S.soft2 = A.soft2;
                S.inv_screen = (A.screen > 0.0 && isfinite(A.screen)) ? 1.0 / A.screen : 0.0;
                keep = true;
                if (HAS_CUT) {
                    const double gx = axis_gap(A.x, lox, hix, perx ? Lx : 0.0);
                    const double gy = axis_gap(A.y, loy, hiy, pery ? Ly : 0.0);
                    const double gz = axis_gap(A.z, loz, hiz, perz ? Lz : 0.0);
                    keep = gx * gx + gy * gy + gz * gz <= rc2;
                }
            }
            if (HAS_CUT) {                                // kept atoms are compacted in list order
                const unsigned ballot = __ballot_sync(0xffffffffu, keep);
                const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
                if (lane == 0) s_warp_count[warp] = __popc(ballot);
                __syncthreads();
                int base = 0;
                na = 0;
#pragma unroll
                for (int w = 0; w < 8; ++w) { if (w < warp) base += s_warp_count[w]; na += s_warp_count[w]; }
                if (keep) s_atoms[base + __popc(ballot & ((1u << lane) - 1u))] = S;
            } else if (keep) {
                s_atoms[threadIdx.x] = S;
            }
        }
        __syncthreads();
        if (!live) continue;
        for (int a = 0; a < na; ++a) {
            const AtomStaged A = s_atoms[a];
            double ddy = y - A.y, ddz = z - A.z;
            if (pery) ddy = fma(-Ly, fma(ddy, iLy, kRoundMagic) - kRoundMagic, ddy);
            if (perz) ddz = fma(-Lz, fma(ddz, iLz, kRoundMagic) - kRoundMagic, ddz);
            // + 1e-200: an atom on a grid point gives r = 1e-100 instead of 0 * inf; any r2 >= 1e-184 is unchanged
            const double yz2 = fma(ddy, ddy, ddz * ddz) + 1e-200;
            const double nZ = -A.Z;
#pragma unroll
            for (int e = 0; e < CELLS; ++e) {
                double ddx = xs[e] - A.x;
                if (perx) ddx = fma(-Lx, fma(ddx, iLx, kRoundMagic) - kRoundMagic, ddx);
                const double r2 = fma(ddx, ddx, yz2);
                double r = sqrt_pos(r2);
                if (HAS_CUT) {
                    // the cutoff is defined on r = sqrt(r2) (correctly rounded): decide on r2 unless it is a tie
                    if (fabs(r2 - rc2) <= 1e-12 * rc2) r = sqrt(r2);
                    if (r > rcut) continue;
                }
                const double screen = exp_nonpositive(-r * A.inv_screen, s_exp2);   // inv_screen = 0: exactly 1
                sum[e] = fma(nZ * screen, rsqrt_pos(r2 + A.soft2), sum[e]);
            }
        }
    }
    if (live) {
#pragma unroll
        for (int e = 0; e < CELLS; ++e) {
            if (i0 + e >= g.nx) continue;
            if (PREFIX_OUT) prefix_out[flat0 + e] = sum[e];
            else store_with_images(V + (long long)blockIdx.y * g.pcells, g, i0 + e, j, k, (real)fmin(fmax(sum[e], vmin), vmax));
        }
    }
}

// Length of the atom-list prefix that every entry shares with entry 0 (compared bit by bit): *out starts at the shortest
// list length and is lowered to the first index at which some entry differs.  grid: x covers min_count, y = batch - 1.
__global__ void common_prefix_kernel(const AtomRec* __restrict__ atoms, const AtomRange* __restrict__ ranges, int min_count,
                                     int* __restrict__ out)
{
    const int a = blockIdx.x * blockDim.x + threadIdx.x;
    if (a >= min_count) return;
    const unsigned long long* p0 = reinterpret_cast<const unsigned long long*>(atoms + ranges[0].first + a);
    const unsigned long long* pb = reinterpret_cast<const unsigned long long*>(atoms + ranges[blockIdx.y + 1].first + a);
    bool same = true;
#pragma unroll
    for (int q = 0; q < 6; ++q) same = same && p0[q] == pb[q];
    if (!same) atomicMin(out, a);
}

// ---------------------------------------------------------------------------------------------
// Potential from a unit-cell grid (PAPER.md:148, 213 step (ii): expansion and interpolation of the DFT potential
// onto the mesh; reading 24): cell[mz][my][mx] doubles at spacings (ax/mx, ay/my, az/(mz-1)), periodic
// in x and y, nearest plane beyond the cell in z, trilinear interpolation at (i dx - x0, j dy - y0, k dz - z0),
// clamp, one rounding to `real`.  The gather hits L1 / L2 (a unit cell is small).
// ---------------------------------------------------------------------------------------------
struct CellParams { int mx, my, mz; double ax, ay, az, x0, y0, z0, vmin, vmax; };

// Block (32, 8): thread (tx, ty) owns the mesh column (i, j) and a z segment of `zs` planes (blockIdx.z): everything that
// depends on x and y only -- the two periodic cell indices and weights per axis, the image offsets of the storage frame -- is
// computed once per column, the march over k keeps the z part.
constexpr int kCellSeg = 32;

template <typename real>
__global__ void __launch_bounds__(256)
potential_cell_kernel(Grid g, double dx, double dy, double dz, const double* __restrict__ cell, CellParams p,
                      real* __restrict__ V /* entry base */)
{
    const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * 8 + threadIdx.y;
    if (i >= g.nx || j >= g.ny) return;
    const int k0 = blockIdx.z * kCellSeg, k1 = min(k0 + kCellSeg, g.nz);
    const double hx = p.ax / p.mx, hy = p.ay / p.my, hz = (p.mz > 1) ? p.az / (p.mz - 1) : 1.0;
    const double u = (i * dx - p.x0) / hx, v = (j * dy - p.y0) / hy;
    const double fu = floor(u), fv = floor(v);
    const double tu = u - fu, tv = v - fv, su = 1.0 - tu, sv = 1.0 - tv;
    // periodic cell index of floor(u): fu - mx * floor(fu / mx), exact in double for any mesh (no 64-bit integer division)
    const int iu0 = (int)(fu - (double)p.mx * floor(fu / (double)p.mx));
    const int iv0 = (int)(fv - (double)p.my * floor(fv / (double)p.my));
    const int iu1 = iu0 + 1 == p.mx ? 0 : iu0 + 1, iv1 = iv0 + 1 == p.my ? 0 : iv0 + 1;
    const int o00 = iv0 * p.mx + iu0, o01 = iv0 * p.mx + iu1, o10 = iv1 * p.mx + iu0, o11 = iv1 * p.mx + iu1;
    const long long cplane = (long long)p.my * p.mx;
    int ix = 0, jy = 0;                  // shifts of the periodic images this column also stores (0: none)
    if (g.bcx == BC_PERIODIC) { if (i < PADX) ix = g.nx; else if (i >= g.nx - PADX) ix = -g.nx; }
    if (g.bcy == BC_PERIODIC) { if (j < PADY) jy = g.ny * g.px; else if (j >= g.ny - PADY) jy = -g.ny * g.px; }
    long long o = cell_offset(g, i, j, k0);
    for (int k = k0; k < k1; ++k, o += g.pplane) {
        const double w = fmin(fmax((k * dz - p.z0) / hz, 0.0), (double)(p.mz - 1));
        const int iw0 = min((int)floor(w), p.mz > 1 ? p.mz - 2 : 0);
        const double tw = (p.mz > 1) ? w - (double)iw0 : 0.0;
        const double* __restrict__ c0p = cell + (long long)iw0 * cplane;
        const double* __restrict__ c1p = (p.mz > 1) ? c0p + cplane : cell;
        // same grouping as the definition: x, then y, then z; products and sums kept separate (no contraction)
        const double c00 = __dadd_rn(__dmul_rn(__ldg(c0p + o00), su), __dmul_rn(__ldg(c0p + o01), tu));
        const double c10 = __dadd_rn(__dmul_rn(__ldg(c0p + o10), su), __dmul_rn(__ldg(c0p + o11), tu));
        const double c01 = __dadd_rn(__dmul_rn(__ldg(c1p + o00), su), __dmul_rn(__ldg(c1p + o01), tu));
        const double c11 = __dadd_rn(__dmul_rn(__ldg(c1p + o10), su), __dmul_rn(__ldg(c1p + o11), tu));
        const double c0 = __dadd_rn(__dmul_rn(c00, sv), __dmul_rn(c10, tv));
        const double c1 = __dadd_rn(__dmul_rn(c01, sv), __dmul_rn(c11, tv));
        const double val = __dadd_rn(__dmul_rn(c0, 1.0 - tw), __dmul_rn(c1, tw));
        const real out = (real)fmin(fmax(val, p.vmin), p.vmax);
        V[o] = out;
        if (ix) V[o + ix] = out;
        if (jy) V[o + jy] = out;
        if (ix && jy) V[o + ix + jy] = out;
    }
}

// ---------------------------------------------------------------------------------------------
// S1 packet init: eq (3) PAPER.md:52 with signed wave vector; staggered start
//   R^0 = Re psi0,  I^{-1/2} = Im psi0 + (1/2) A Re psi0,  A f = -c d2 f + c_v V f   (reading 4)
// evaluated in double from the stored V; neighbours of Re psi0 are re-evaluated analytically at the
// (wrapped) neighbour grid point, or are 0 beyond a Dirichlet face.
// ---------------------------------------------------------------------------------------------
struct PacketParams { double x0, y0, z0, inv2s2, kx, ky, kz, amp; };
struct Mesh { double dx, dy, dz; double cx, cy, cz, cv; };   // spacings and the coefficients of PAPER.md:87

__device__ __forceinline__ void packet_eval(const PacketParams& p, const Mesh& m, int i, int j, int k,
                                            double* re, double* im)
{
    const double ddx = i * m.dx - p.x0, ddy = j * m.dy - p.y0, ddz = k * m.dz - p.z0;
    const double G = p.amp * exp(-(ddx * ddx + ddy * ddy + ddz * ddz) * p.inv2s2);
    const double phi = p.kx * ddx + p.ky * ddy + p.kz * ddz;
    double s, c;
    sincos(phi, &s, &c);
    *re = G * c;
    *im = G * s;
}

__device__ __forceinline__ double packet_re_nbr(const PacketParams& p, const Grid& g, const Mesh& m,
                                                int i, int j, int k)
{
    if (i < 0 || i >= g.nx) { if (g.bcx == BC_PERIODIC) i = wrap_index(i, g.nx); else return 0.0; }
    if (j < 0 || j >= g.ny) { if (g.bcy == BC_PERIODIC) j = wrap_index(j, g.ny); else return 0.0; }
    if (k < 0 || k >= g.nz) { if (g.bcz == BC_PERIODIC) k = wrap_index(k, g.nz); else return 0.0; }
    double re, im;
    packet_eval(p, m, i, j, k, &re, &im);
    return re;
}

template <typename real>
__global__ void __launch_bounds__(256)
wavepacket_init_kernel(Grid g, Mesh m, PacketParams p, int nent /* entries that get this packet, consecutive */,
                       const real* __restrict__ V, real* __restrict__ R, real* __restrict__ I)
{
    const long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (cell >= g.cells) return;
    const int i = (int)(cell % g.nx);
    const long long t = cell / g.nx;
    const int j = (int)(t % g.ny);
    const int k = (int)(t / g.ny);
    double re, im;
    packet_eval(p, m, i, j, k, &re, &im);
    const double d2x = packet_re_nbr(p, g, m, i + 1, j, k) - 2.0 * re + packet_re_nbr(p, g, m, i - 1, j, k);
    const double d2y = packet_re_nbr(p, g, m, i, j + 1, k) - 2.0 * re + packet_re_nbr(p, g, m, i, j - 1, k);
    const double d2z = packet_re_nbr(p, g, m, i, j, k + 1) - 2.0 * re + packet_re_nbr(p, g, m, i, j, k - 1);
    const double kin = -m.cx * d2x - m.cy * d2y - m.cz * d2z;
    const long long o = cell_offset(g, i, j, k);
    // the packet is the same for every entry; only the potential term of the staggered start differs
    for (int e = 0; e < nent; ++e) {
        const long long eo = (long long)e * g.pcells;
        const double Ar = kin + m.cv * (double)V[eo + o] * re;
        store_with_images(R + eo, g, i, j, k, (real)re);
        store_with_images(I + eo, g, i, j, k, (real)(im + 0.5 * Ar));
    }
}

// ---------------------------------------------------------------------------------------------
// Two-pass reference stencil: one thread per cell, neighbours straight from global memory (L1/L2).
//   sgn = +1: eq (9) PAPER.md:83  dst = I, src = R;   sgn = -1: eq (8) PAPER.md:74  dst = R, src = I
//   dst <- M[k] * ( dst + sgn * ( c_x d2x(src) + c_y d2y(src) + c_z d2z(src) - c_v V src ) )
// In place is safe (dst is read only at the thread's own cell).  Works for every shape and boundary
// combination; the fused kernels in tdse_kernels_fused.cuh are the fast path.
// ---------------------------------------------------------------------------------------------
template <typename real>
__device__ __forceinline__ real load_nbr(const real* __restrict__ f, const Grid& g, int i, int j, int k)
{
    if (i < 0)     { if (g.bcx == BC_PERIODIC) i = g.nx - 1; else return (real)0; }
    if (i >= g.nx) { if (g.bcx == BC_PERIODIC) i = 0;        else return (real)0; }
    if (j < 0)     { if (g.bcy == BC_PERIODIC) j = g.ny - 1; else return (real)0; }
    if (j >= g.ny) { if (g.bcy == BC_PERIODIC) j = 0;        else return (real)0; }
    if (k < 0)     { if (g.bcz == BC_PERIODIC) k = g.nz - 1; else return (real)0; }
    if (k >= g.nz) { if (g.bcz == BC_PERIODIC) k = 0;        else return (real)0; }
    return f[cell_offset(g, i, j, k)];
}

// Block (32, 8): thread (tx, ty) owns the column (i, j) = (32 bx + tx, 8 by + ty) of one entry and marches a z segment
// of `zs` planes, keeping the z neighbours of the source field in registers.  Neighbour offsets follow eqs (13)-(14)
// (wrap on a periodic axis, zero beyond a Dirichlet face) and are fixed per column, so the loop has no index
// arithmetic; the storage frame is written (store_with_images) but not relied on: domains narrower than two frames take this path.
// grid: x = ceil(nx / 32), y = ceil(ny / 8), z = batch * nseg.  In place: a cell's update reads only its own dst.
template <typename real>
__global__ void __launch_bounds__(256)
half_step_kernel(Grid g, real cx, real cy, real cz, real cv, real sgn, int zs, int nseg, const real* __restrict__ V,
                 const real* __restrict__ M, const real* __restrict__ src, real* __restrict__ dst)
{
    const int i = blockIdx.x * 32 + threadIdx.x, j = blockIdx.y * 8 + threadIdx.y;
    if (i >= g.nx || j >= g.ny) return;
    const int b = blockIdx.z / nseg, seg = blockIdx.z % nseg;
    const int k0 = seg * zs, k1 = min(k0 + zs, g.nz);
    const long long base = (long long)b * g.pcells;
    const real* __restrict__ s = src + base;
    const real* __restrict__ v = V + base;
    real* __restrict__ d = dst + base;
    int ix = 0, jy = 0;                  // shifts of the periodic images this column also stores (0: none)
    if (g.bcx == BC_PERIODIC) { if (i < PADX) ix = g.nx; else if (i >= g.nx - PADX) ix = -g.nx; }
    if (g.bcy == BC_PERIODIC) { if (j < PADY) jy = g.ny * g.px; else if (j >= g.ny - PADY) jy = -g.ny * g.px; }
    auto plane_value = [&](int k) -> real {        // source value of this column at plane k, any k in [-1, nz]
        if (k < 0)     { if (g.bcz == BC_PERIODIC) k = g.nz - 1; else return (real)0; }
        if (k >= g.nz) { if (g.bcz == BC_PERIODIC) k = 0;        else return (real)0; }
        return s[cell_offset(g, i, j, k)];
    };
    // x/y neighbour offsets relative to the cell, and whether the neighbour exists (else: Dirichlet zero)
    const bool vxl = i > 0 || g.bcx == BC_PERIODIC, vxh = i < g.nx - 1 || g.bcx == BC_PERIODIC;
    const bool vyl = j > 0 || g.bcy == BC_PERIODIC, vyh = j < g.ny - 1 || g.bcy == BC_PERIODIC;
    const int oxl = i > 0 ? -1 : g.nx - 1, oxh = i < g.nx - 1 ? 1 : 1 - g.nx;
    const int oyl = (j > 0 ? -1 : g.ny - 1) * g.px, oyh = (j < g.ny - 1 ? 1 : 1 - g.ny) * g.px;
    real zlo = plane_value(k0 - 1), s0 = plane_value(k0);
    long long o = cell_offset(g, i, j, k0);
    for (int k = k0; k < k1; ++k, o += g.pplane) {
        const real zhi = plane_value(k + 1);
        const real xh = vxh ? s[o + oxh] : (real)0, xl = vxl ? s[o + oxl] : (real)0;
        const real yh = vyh ? s[o + oyh] : (real)0, yl = vyl ? s[o + oyl] : (real)0;
        const real d2x = (xh + xl) - (real)2 * s0;
        const real d2y = (yh + yl) - (real)2 * s0;
        const real d2z = (zhi + zlo) - (real)2 * s0;
        const real upd = cx * d2x + cy * d2y + cz * d2z - cv * v[o] * s0;
        const real out = M[k] * (d[o] + sgn * upd);
        d[o] = out;
        if (ix) d[o + ix] = out;
        if (jy) d[o + jy] = out;
        if (ix && jy) d[o + ix + jy] = out;
        zlo = s0; s0 = zhi;
    }
}

// ---------------------------------------------------------------------------------------------
// S5 detector (eq (15), density of PAPER.md:87): D += R^2 + I^2 on plane k_det and
// trace[b][slot] = scale * sum of the plane (scale = dx dy), in ONE launch per sample: warp-shuffle block sums go
// to partial[b][block]; the block that finishes last for an entry (a counter per entry, reset for the next sample)
// adds the partials serially in block order, so the sum does not depend on which block that was.  Frame mode
// (the trajectory rho = {rho(0), rho(h dt), ...}) also keeps the sampled plane: frame[b][p] = rho.
// D, partial and frame may each be NULL (frame-only call for rho(0)).  grid: x = ceil(nx*ny / 256), y = batch.
// Launched with programmatic stream serialization behind the fused step kernel: nothing global is touched before
// griddepcontrol.wait.
// ---------------------------------------------------------------------------------------------
template <typename real>
__global__ void __launch_bounds__(256)
detector_accum_kernel(Grid g, int k_det, const real* __restrict__ R, const real* __restrict__ I,
                      double* __restrict__ D, double* __restrict__ partial /* [batch][gridDim.x] */,
                      double* __restrict__ frame /* this sample's frame of entry 0 */, long long frame_entry_stride,
                      unsigned* __restrict__ done /* [batch] */, double scale, double* __restrict__ trace,
                      int max_samples, int slot)
{
    __shared__ double scratch[32];
    asm volatile("griddepcontrol.wait;\n" ::: "memory");
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    double rho = 0.0;
    if (p < g.plane) {
        const long long off = (long long)blockIdx.y * g.pcells + cell_offset(g, (int)(p % g.nx), (int)(p / g.nx), k_det);
        const double r = (double)R[off], im = (double)I[off];
        rho = r * r + im * im;
        if (D) D[(long long)blockIdx.y * g.plane + p] += rho;
        if (frame) frame[(long long)blockIdx.y * frame_entry_stride + p] = rho;
    }
    if (partial) {
        const double s = block_sum(rho, scratch);
        if (threadIdx.x == 0) {
            double* part = partial + (long long)blockIdx.y * gridDim.x;
            part[blockIdx.x] = s;
            __threadfence();                                  // the partial is visible before the count
            const unsigned before = atomicAdd(done + blockIdx.y, 1u);
            if (before == gridDim.x - 1) {                    // every block of this entry has published its partial
                __threadfence();
                double t = 0.0;
                for (unsigned q = 0; q < gridDim.x; ++q) t += __ldcg(part + q);   // fixed order; L2, not a stale L1 line
                if (slot < max_samples) trace[(long long)blockIdx.y * max_samples + slot] = scale * t;
                done[blockIdx.y] = 0;                         // ready for the next sample (same stream: ordered)
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Trajectory dissimilarity, eq (16), over the batch entries of one context:
//   d_kj = mean over frames s0..s1 of sqrt( dA * sum_p (rho_k[s][p] - rho_j[s][p])^2 )      (reading 23)
// A block takes a kDisTile x kDisTile tile of entry pairs and one frame, so every frame it reads serves
// kDisTile pairs (64 fp64 accumulators per thread: 1 flop per byte read, so the pass stays memory-bound); fixed-order block sums (deterministic).  inner[(k*batch + j)*nwin + s-s0] = sqrt(dA * sum).
// grid: x = tiles_k * tiles_j, y = nwin.
// ---------------------------------------------------------------------------------------------
constexpr int kDisTile = 8;

__global__ void __launch_bounds__(256)
dissimilarity_inner_kernel(const double* __restrict__ frames, int batch, long long entry_stride, int npix,
                           double dA, int s0, int nwin, double* __restrict__ inner)
{
    __shared__ double scratch[32];
    const int tiles = (batch + kDisTile - 1) / kDisTile;
    const int tk = blockIdx.x / tiles, tj = blockIdx.x % tiles;
    if (tj < tk) return;                              // d is symmetric: upper triangle of tiles only
    const int s = blockIdx.y;
    const double* fk[kDisTile];
    const double* fj[kDisTile];
#pragma unroll
    for (int q = 0; q < kDisTile; ++q) {
        fk[q] = frames + (long long)min(tk * kDisTile + q, batch - 1) * entry_stride + (long long)(s0 + s) * npix;
        fj[q] = frames + (long long)min(tj * kDisTile + q, batch - 1) * entry_stride + (long long)(s0 + s) * npix;
    }
    double acc[kDisTile][kDisTile];
#pragma unroll
    for (int a = 0; a < kDisTile; ++a)
#pragma unroll
        for (int b = 0; b < kDisTile; ++b) acc[a][b] = 0.0;
    for (int p = threadIdx.x; p < npix; p += blockDim.x) {
        double vk[kDisTile], vj[kDisTile];
#pragma unroll
        for (int q = 0; q < kDisTile; ++q) { vk[q] = fk[q][p]; vj[q] = fj[q][p]; }
#pragma unroll
        for (int a = 0; a < kDisTile; ++a)
#pragma unroll
            for (int b = 0; b < kDisTile; ++b) { const double d = vk[a] - vj[b]; acc[a][b] = fma(d, d, acc[a][b]); }
    }
#pragma unroll
    for (int a = 0; a < kDisTile; ++a)
#pragma unroll
        for (int b = 0; b < kDisTile; ++b) {
            const double t = block_sum(acc[a][b], scratch);
            const int k = tk * kDisTile + a, j = tj * kDisTile + b;
            if (threadIdx.x == 0 && k < batch && j < batch)
                inner[((long long)k * batch + j) * nwin + s] = sqrt(dA * t);
        }
}

// d[k][j] = d[j][k] = mean_s inner[k][j][s] for k <= j (serial over frames, fixed order).  One thread per pair.
__global__ void dissimilarity_finish_kernel(const double* __restrict__ inner, int batch, int nwin, double* __restrict__ d)
{
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= batch * batch) return;
    const int k = q / batch, j = q % batch;
    if (j < k) return;
    double acc = 0.0;
    for (int s = 0; s < nwin; ++s) acc += inner[((long long)k * batch + j) * nwin + s];
    const double v = (k == j) ? 0.0 : acc / (double)nwin;
    d[(long long)k * batch + j] = v;
    d[(long long)j * batch + k] = v;
}

// ---------------------------------------------------------------------------------------------
// Diagnostics: q_paper = sum R^2 + I^2, q_visscher = sum R^2 + I(+) I with a look-ahead eq (9) in double.
// One entry at a time; per-block partials [2][gridDim.x]; reduce_pairs_kernel finishes.
// ---------------------------------------------------------------------------------------------
template <typename real>
__global__ void __launch_bounds__(256)
norm_partial_kernel(Grid g, Mesh m, const real* __restrict__ V, const real* __restrict__ M,
                    const real* __restrict__ R, const real* __restrict__ I, double* __restrict__ partial)
{
    __shared__ double scratch[32];
    const long long cell = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    double qv = 0.0, qp = 0.0;
    if (cell < g.cells) {
        const int i = (int)(cell % g.nx);
        const long long t = cell / g.nx;
        const int j = (int)(t % g.ny);
        const int k = (int)(t / g.ny);
        const long long o = cell_offset(g, i, j, k);
        const double r0 = (double)R[o], i0 = (double)I[o];
        const double d2x = ((double)load_nbr(R, g, i + 1, j, k) + (double)load_nbr(R, g, i - 1, j, k)) - 2.0 * r0;
        const double d2y = ((double)load_nbr(R, g, i, j + 1, k) + (double)load_nbr(R, g, i, j - 1, k)) - 2.0 * r0;
        const double d2z = ((double)load_nbr(R, g, i, j, k + 1) + (double)load_nbr(R, g, i, j, k - 1)) - 2.0 * r0;
        const double ip = (double)M[k] * (i0 + m.cx * d2x + m.cy * d2y + m.cz * d2z - m.cv * (double)V[o] * r0);
        qv = r0 * r0 + ip * i0;
        qp = r0 * r0 + i0 * i0;
    }
    const double sv = block_sum(qv, scratch);
    const double sp = block_sum(qp, scratch);
    if (threadIdx.x == 0) {
        partial[blockIdx.x] = sv;
        partial[gridDim.x + blockIdx.x] = sp;
    }
}

// out[r] = scale * sum_q partial[r*n + q], r = 0..rows-1; single block, fixed order per thread stripe.
__global__ void __launch_bounds__(256)
reduce_rows_kernel(const double* __restrict__ partial, int n, int rows, double scale, double* __restrict__ out)
{
    __shared__ double scratch[32];
    for (int r = 0; r < rows; ++r) {
        double s = 0.0;
        for (int q = threadIdx.x; q < n; q += blockDim.x) s += partial[(long long)r * n + q];
        s = block_sum(s, scratch);
        if (threadIdx.x == 0) out[r] = scale * s;
    }
}

// Fill the frame of one entry's array with the periodic images of the interior (after a raw upload).
// One thread per stored element of the entry; Dirichlet axes keep their zero frame.
template <typename real>
__global__ void __launch_bounds__(256)
frame_fill_kernel(Grid g, real* __restrict__ f)
{
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= g.pcells) return;
    const int xi = (int)(e % g.px) - PADX;
    const long long t = e / g.px;
    const int yj = (int)(t % g.py) - PADY;
    const int k = (int)(t / g.py);
    const bool fx = xi < 0 || xi >= g.nx, fy = yj < 0 || yj >= g.ny;
    if (!fx && !fy) return;
    if ((fx && g.bcx != BC_PERIODIC) || (fy && g.bcy != BC_PERIODIC)) { f[e] = (real)0; return; }
    f[e] = f[cell_offset(g, wrap_index(xi, g.nx), wrap_index(yj, g.ny), k)];
}

// max |V| over one entry (for the stability bound after a raw-grid upload).  The frame holds images or zeros,
// so scanning the stored elements gives the same maximum.
template <typename real>
__global__ void __launch_bounds__(256)
absmax_partial_kernel(const real* __restrict__ V, long long n, double* __restrict__ partial)
{
    __shared__ double s_max[256];
    double m = 0.0;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (long long)gridDim.x * blockDim.x)
        m = fmax(m, fabs((double)V[q]));
    s_max[threadIdx.x] = m;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) s_max[threadIdx.x] = fmax(s_max[threadIdx.x], s_max[threadIdx.x + o]);
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = s_max[0];
}

__global__ void fill_zero_kernel(double* p, long long n)
{
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += (long long)gridDim.x * blockDim.x)
        p[q] = 0.0;
}

}  // namespace tdse
