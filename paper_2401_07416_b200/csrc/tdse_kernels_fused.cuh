// tdse_kernels_fused.cuh -- the fused, temporally blocked FDTD step for sm_100a.
//
// One launch advances every batch entry by T full time steps = 2T half-steps ("stages"):
//   stage 2m+1: I^{n+m+1/2} = M[k] * ( I^{n+m-1/2} + ( c * lap(R^{n+m})     - (6c + c_v V) R^{n+m}     ) )   eq (9)
//   stage 2m+2: R^{n+m+1}   = M[k] * ( R^{n+m}     - ( c * lap(I^{n+m+1/2}) - (6c + c_v V) I^{n+m+1/2} ) )   eq (8)
// where lap(f) = sum of the 6 neighbours (the -6 f of the three second differences is folded into the
// diagonal), boundary handling per eqs (13)-(14) PAPER.md:126-136 (periodic) or zero-Dirichlet, and the
// absorbing mask M[k] (eq (10) PAPER.md:89-94 as a polynomial mask) fused into the same pass.
//
// Design (differs from the paper's one-thread-per-point kernel, on purpose):
//   * a CTA owns an xy tile (BX x BY cells + halo of 2T) of one batch entry and marches a z chunk;
//     ping-pong buffers (Rin,Iin -> Rout,Iout) make neighbouring tiles independent;
//   * planes of R, I, V arrive in a shared-memory ring through cp.async (16 B per thread, zero fill
//     for Dirichlet ghosts, index wrap for periodic axes resolved once per thread before the march);
//   * each thread keeps, per stage, the previous two z-planes of its cells in registers (register-rotated
//     z neighbours); y neighbours come from a double-buffered shared-memory plane per stage, x neighbours
//     from warp shuffles (lane edges read shared memory);
//   * all 2T stages of the software pipeline run between two __syncthreads(); stage s works on plane p-s
//     while plane p+PF is in flight;
//   * final R and I planes are written with 128-bit stores; on a sampling step the CTAs that own the
//     detector plane add R^2 + I^2 into the image and produce one partial sum per tile (warp-shuffle
//     reduction) for the trace.
// Compulsory HBM traffic: 5 words per cell per launch, i.e. 5/T words per cell-update.
#pragma once
#include "tdse_common.cuh"

namespace tdse {

struct FusedParams {
    const void* Rin; const void* Iin; const void* V;   // [batch][nz][ny][nx]
    void* Rout; void* Iout;
    const void* mask;                                  // real[nz]
    int nx, ny, nz, batch;
    int bcx, bcy, bcz;
    int tiles_x, tiles_y, nchunks, bz;                 // z chunk length (last chunk may be shorter)
    double c, cv;
    int sample;                                        // 1: accumulate detector on plane k_det
    int k_det;
    double* D;                                         // [batch][ny][nx]
    double* partial;                                   // [batch][tiles_x*tiles_y]
};

__device__ __forceinline__ void cp_async_16(void* smem_dst, const void* gmem_src, int src_bytes)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(s), "l"(gmem_src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory"); }

template <typename real, int T_, int BX_, int BY_, int NT_, int PF_>
struct FusedTraits {
    static constexpr int T = T_, BX = BX_, BY = BY_, NT = NT_, PF = PF_;
    static constexpr int VW = 16 / sizeof(real);
    static constexpr int NS = 2 * T;                           // stages per launch
    static constexpr int H = 2 * T;                            // halo (cells) in y, planes in z
    static constexpr int HX = ((2 * T + VW - 1) / VW) * VW;    // halo in x, vector aligned
    static constexpr int W = BX + 2 * HX;
    static constexpr int RH = BY + 2 * H;
    static constexpr int WQ = W / VW;                          // 16-byte groups per row
    static constexpr int G = WQ * RH;                          // groups per plane
    static constexpr int GPT = (G + NT - 1) / NT;              // groups per thread
    static constexpr int PLANE = W * RH;                       // elements per staged plane
    static constexpr int RD = PF + 2;                          // ring depth
    static constexpr int SMEM_ELEMS = 3 * RD * PLANE + (NS - 1) * 2 * PLANE;
    static constexpr size_t SMEM_BYTES = (size_t)SMEM_ELEMS * sizeof(real) + 32 * sizeof(double);
    static_assert(BX % VW == 0, "tile width must be a multiple of the vector width");
    static_assert(NT % 32 == 0, "whole warps");
};

template <typename real, int T, int BX, int BY, int NT, int PF>
__global__ void __launch_bounds__(NT, 1)
fdtd_fused_kernel(const FusedParams P)
{
    using Tr = FusedTraits<real, T, BX, BY, NT, PF>;
    using V4 = Pack<real>;
    constexpr int VW = Tr::VW, NS = Tr::NS, H = Tr::H, HX = Tr::HX, WQ = Tr::WQ, RH = Tr::RH;
    constexpr int G = Tr::G, GPT = Tr::GPT, PLANE = Tr::PLANE, RD = Tr::RD;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    real* const ringR = reinterpret_cast<real*>(smem_raw);
    real* const ringI = ringR + RD * PLANE;
    real* const ringV = ringI + RD * PLANE;
    real* const exch = ringV + RD * PLANE;                 // [(NS-1)][2][PLANE], stage s output at exch[(s-1)*2 + parity]
    double* const scratch = reinterpret_cast<double*>(exch + (NS - 1) * 2 * PLANE);

    const int tid = threadIdx.x, lane = tid & 31;
    const int ntiles = P.tiles_x * P.tiles_y;
    int bid = blockIdx.x;
    const int tile = bid % ntiles; bid /= ntiles;
    const int chunk = bid % P.nchunks;
    const int b = bid / P.nchunks;
    const int X0 = (tile % P.tiles_x) * BX, Y0 = (tile / P.tiles_x) * BY;
    const int Z0 = chunk * P.bz;
    const int bzc = min(P.bz, P.nz - Z0);
    const long long plane = (long long)P.nx * P.ny;
    const long long ebase = (long long)b * plane * P.nz;

    const real* __restrict__ gR = static_cast<const real*>(P.Rin) + ebase;
    const real* __restrict__ gI = static_cast<const real*>(P.Iin) + ebase;
    const real* __restrict__ gV = static_cast<const real*>(P.V) + ebase;
    real* __restrict__ oR = static_cast<real*>(P.Rout) + ebase;
    real* __restrict__ oI = static_cast<real*>(P.Iout) + ebase;
    const real* __restrict__ gM = static_cast<const real*>(P.mask);

    const real c = (real)P.c, cv = (real)P.cv, c6 = (real)(6.0 * P.c);

    // ---- per-thread geometry, fixed for the whole march ---------------------------------------
    int  goff[GPT];      // offset of the group inside a plane (wrapped), elements
    int  soff[GPT];      // offset inside a staged plane, elements
    bool ldok[GPT];      // load from memory (else zero fill: Dirichlet ghost / inactive)
    bool core[GPT];      // group belongs to the tile's own cells and lies inside the domain
    int  row[GPT];
#pragma unroll
    for (int j = 0; j < GPT; ++j) {
        const int g = tid + j * NT;
        const bool act = g < G;
        const int r = act ? g / WQ : 0, q = act ? g % WQ : 0;
        row[j] = act ? r : -1000;
        soff[j] = (act ? g : 0) * VW;
        const int xg = X0 - HX + q * VW, yg = Y0 - H + r;
        bool inx = xg >= 0 && xg < P.nx, iny = yg >= 0 && yg < P.ny;
        int xw = xg, yw = yg;
        if (P.bcx == BC_PERIODIC) { xw = wrap_index(xg, P.nx); inx = true; }
        if (P.bcy == BC_PERIODIC) { yw = wrap_index(yg, P.ny); iny = true; }
        ldok[j] = act && inx && iny;
        goff[j] = ldok[j] ? yw * P.nx + xw : 0;
        core[j] = act && q * VW >= HX && q * VW < HX + BX && r >= H && r < H + BY &&
                  xg < P.nx && yg < P.ny;   // xg, yg >= 0 is implied for core groups
    }

    auto zplane = [&](int pz, bool& ok) -> int {     // global plane index -> (wrapped index, loadable?)
        ok = pz >= 0 && pz < P.nz;
        if (P.bcz == BC_PERIODIC) { ok = true; return wrap_index(pz, P.nz); }
        return ok ? pz : 0;
    };
    auto issue_plane = [&](int t) {                  // stage plane t of the march into ring slot t % RD
        bool zok;
        const int pz = zplane(Z0 - H + t, zok);
        const long long poff = (long long)pz * plane;
        const int slot = (t % RD) * PLANE;
#pragma unroll
        for (int j = 0; j < GPT; ++j) {
            if (tid + j * NT < G) {
                const int nbytes = (ldok[j] && zok) ? 16 : 0;
                const long long o = poff + goff[j];
                cp_async_16(ringR + slot + soff[j], gR + o, nbytes);
                cp_async_16(ringI + slot + soff[j], gI + o, nbytes);
                cp_async_16(ringV + slot + soff[j], gV + o, nbytes);
            }
        }
    };

    // ---- register queues ------------------------------------------------------------------------
    // f[s] (s = 0..NS-1): field after stage s (s = 0: R as loaded).  mid = plane p-s-1, old = plane p-s-2
    // relative to the plane p that arrives in the current iteration.
    V4 fmid[NS][GPT], fold[NS][GPT];
    V4 vq[NS + 1][GPT];      // vq[s] = 6c + c_v V at plane p-s, s = 2..NS (index 0, 1 unused)
    real mq[NS + 1];         // mq[s] = mask of plane p-s
#pragma unroll
    for (int s = 0; s < NS; ++s)
#pragma unroll
        for (int j = 0; j < GPT; ++j)
#pragma unroll
            for (int e = 0; e < VW; ++e) { fmid[s][j].e[e] = 0; fold[s][j].e[e] = 0; }
#pragma unroll
    for (int s = 0; s <= NS; ++s) {
        mq[s] = 0;
#pragma unroll
        for (int j = 0; j < GPT; ++j)
#pragma unroll
            for (int e = 0; e < VW; ++e) vq[s][j].e[e] = 0;
    }
    // exchange planes start defined (they are read one iteration before they are first written)
    for (int q = tid; q < (NS - 1) * 2 * PLANE; q += NT) exch[q] = 0;

    double det_sum = 0.0;
    const int niter = bzc + 2 * H;                   // planes Z0-H .. Z0+bzc+H-1

    // ---- prologue: PF planes in flight -----------------------------------------------------------
#pragma unroll
    for (int t = 0; t < PF; ++t) { if (t < niter) issue_plane(t); cp_async_commit(); }

#pragma unroll 1
    for (int t = 0; t < niter; ++t) {
        cp_async_wait<PF - 1>();
        __syncthreads();
        if (t + PF < niter) issue_plane(t + PF);
        cp_async_commit();

        const int p = Z0 - H + t;                    // global plane that just arrived
        const int cur = (t % RD) * PLANE;
        const int prv = ((t + RD - 1) % RD) * PLANE;
        const int par = t & 1;
        // mask of plane p-1 enters the queue (0 outside a Dirichlet domain -> forces ghost planes to zero)
#pragma unroll
        for (int s = NS; s > 1; --s) mq[s] = mq[s - 1];
        {
            bool zok;
            const int pz = zplane(p - 1, zok);
            mq[1] = zok ? gM[pz] : (real)0;
        }

#pragma unroll
        for (int j = 0; j < GPT; ++j) {
            const bool act = tid + j * NT < G;       // inactive tail groups still take part in the shuffles
            V4 fnew[NS + 1];
            fnew[0] = *reinterpret_cast<const V4*>(ringR + cur + soff[j]);
            const V4 iold = *reinterpret_cast<const V4*>(ringI + prv + soff[j]);
            const V4 vraw = *reinterpret_cast<const V4*>(ringV + prv + soff[j]);
            V4 dg1;
#pragma unroll
            for (int e = 0; e < VW; ++e) dg1.e[e] = fma(cv, vraw.e[e], c6);

#pragma unroll
            for (int s = 1; s <= NS; ++s) {
                const V4& ctr = fmid[s - 1][j];
                const V4& zlo = fold[s - 1][j];
                const V4& zhi = fnew[s - 1];
                const V4& older = (s == 1) ? iold : fold[s >= 2 ? s - 2 : 0][j];
                const V4& dg = (s == 1) ? dg1 : vq[s][j];
                // plane holding the centre values of this stage (written by the previous iteration)
                const real* cplane = (s == 1) ? (ringR + prv) : (exch + ((s >= 2 ? s - 2 : 0) * 2 + (par ^ 1)) * PLANE);
                // x neighbours: shuffles inside the warp, shared memory at the warp edges
                real xm = __shfl_up_sync(0xffffffffu, ctr.e[VW - 1], 1);
                real xp = __shfl_down_sync(0xffffffffu, ctr.e[0], 1);
                const bool rowok = row[j] >= s && row[j] < RH - s;
                V4 out;
                if (rowok) {
                    if (lane == 0) xm = cplane[soff[j] - 1];
                    if (lane == 31) xp = cplane[soff[j] + VW];
                    const V4 ym = *reinterpret_cast<const V4*>(cplane + soff[j] - WQ * VW);
                    const V4 yp = *reinterpret_cast<const V4*>(cplane + soff[j] + WQ * VW);
                    const real m = ldok[j] ? mq[s] : (real)0;
                    const real sg = (s & 1) ? (real)1 : (real)-1;
#pragma unroll
                    for (int e = 0; e < VW; ++e) {
                        const real left = (e == 0) ? xm : ctr.e[e - 1];
                        const real right = (e == VW - 1) ? xp : ctr.e[e + 1];
                        const real nb = ((left + right) + (ym.e[e] + yp.e[e])) + (zlo.e[e] + zhi.e[e]);
                        const real upd = fma(c, nb, -dg.e[e] * ctr.e[e]);
                        out.e[e] = m * fma(sg, upd, older.e[e]);
                    }
                } else {
#pragma unroll
                    for (int e = 0; e < VW; ++e) out.e[e] = 0;
                }
                fnew[s] = out;
                if (s < NS && act) *reinterpret_cast<V4*>(exch + ((s - 1) * 2 + par) * PLANE + soff[j]) = out;

                // ---- final stages: write back -----------------------------------------------------
                if (s == NS - 1) {                   // I^{n+T-1/2} at plane p-NS+1
                    const int pz = p - (NS - 1);
                    if (core[j] && pz >= Z0 && pz < Z0 + bzc)
                        *reinterpret_cast<V4*>(oI + (long long)pz * plane + goff[j]) = out;
                }
                if (s == NS) {                       // R^{n+T} at plane p-NS
                    const int pz = p - NS;
                    if (core[j] && pz >= Z0 && pz < Z0 + bzc) {
                        *reinterpret_cast<V4*>(oR + (long long)pz * plane + goff[j]) = out;
                        if (P.sample && pz == P.k_det) {
                            // density of PAPER.md:87: (R^s)^2 + (I^{s-1/2})^2; I at this plane is the centre of stage NS
                            double* Dp = P.D + (long long)b * plane + goff[j];
#pragma unroll
                            for (int e = 0; e < VW; ++e) {
                                const double r = (double)out.e[e], im = (double)ctr.e[e];
                                const double rho = r * r + im * im;
                                Dp[e] += rho;
                                det_sum += rho;
                            }
                        }
                    }
                }
            }
            // ---- rotate the z queues (old <- mid <- new) and the diagonal queue -----------------------
#pragma unroll
            for (int s = 0; s < NS; ++s) { fold[s][j] = fmid[s][j]; fmid[s][j] = fnew[s]; }
#pragma unroll
            for (int s = NS; s > 2; --s) vq[s][j] = vq[s - 1][j];
            vq[2][j] = dg1;
        }
    }
    cp_async_wait<0>();

    if (P.sample && P.k_det >= Z0 && P.k_det < Z0 + bzc) {
        const double s = block_sum(det_sum, scratch);
        if (tid == 0) P.partial[(long long)b * ntiles + tile] = s;
    }
}

}  // namespace tdse
