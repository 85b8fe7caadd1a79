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
//     z neighbours: the march is unrolled by 3 so the rotation costs no moves); y neighbours come from a
//     double-buffered shared-memory plane per stage, x neighbours from warp shuffles (lane edges read
//     shared memory);
//   * all 2T stages of the software pipeline run between two __syncthreads(); stage s works on plane p-s
//     while plane p+PF is in flight;
//   * halo cells are recomputed, not exchanged: the region shrinks by one cell per stage, and values
//     outside that shrinking region are garbage that never reaches a cell that is stored.
// Compulsory HBM traffic: 5 words per cell per launch, i.e. 5/T words per cell-update.
#pragma once
#include <type_traits>

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
    static constexpr int PS = GPT * NT * VW;                   // plane stride in shared memory (padded to whole threads)
    static constexpr int GUARD = W;                            // one row before the first and after the last plane
    static constexpr int RD = PF + 2;                          // ring depth
    static constexpr int XD = 3;                               // exchange planes per stage (period of the unrolled march)
    static constexpr int NPLANES = 3 * RD + (NS - 1) * XD;
    static constexpr size_t SMEM_FIXED = ((size_t)NPLANES * PS + 2 * GUARD) * sizeof(real);
    // + (bz + 2H + 2) mask values, added by the launcher
    static_assert(BX % VW == 0, "tile width must be a multiple of the vector width");
    static_assert(NT % 32 == 0, "whole warps");
    static_assert(T == 1 || T == 2, "queue rotation below is written for T = 1, 2");
    static_assert(RD == 3, "ring slots are compile-time constants of the 3x unrolled march");
};

template <typename real, int NS, int GPT>
struct Queue {                       // one z-plane worth of per-thread pipeline state
    Pack<real> f[NS][GPT];           // f[s]: field after stage s (s = 0: R as loaded)
    Pack<real> dg[GPT];              // 6c + c_v V of the plane that entered together with f[0]
};

template <typename real, int T, int BX, int BY, int NT, int PF>
__global__ void __launch_bounds__(NT, 1)
fdtd_fused_kernel(const FusedParams P)
{
    using Tr = FusedTraits<real, T, BX, BY, NT, PF>;
    using V4 = Pack<real>;
    using Q = Queue<real, Tr::NS, Tr::GPT>;
    constexpr int VW = Tr::VW, NS = Tr::NS, H = Tr::H, HX = Tr::HX, WQ = Tr::WQ;
    constexpr int G = Tr::G, GPT = Tr::GPT, PS = Tr::PS, RD = Tr::RD, XD = Tr::XD;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    real* const ringR = reinterpret_cast<real*>(smem_raw) + Tr::GUARD;
    real* const ringI = ringR + RD * PS;
    real* const ringV = ringI + RD * PS;
    real* const exch = ringV + RD * PS;                    // stage s output of iteration t at exch[((s-1)*XD + t%3) * PS]
    real* const smask = exch + (NS - 1) * XD * PS + Tr::GUARD;  // smask[q] = mask of plane Z0-H-1+q

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
    const int soff0 = tid * VW;                      // group j of this thread sits at soff0 + j*NT*VW
    const int edge_off = (lane == 31) ? VW : -lane * VW - 1;   // see the x-neighbour load in body()

    // ---- per-thread geometry, fixed for the whole march ---------------------------------------
    int  goff[GPT];      // offset of the group inside a plane (wrapped), elements
    bool ldok[GPT];      // load from memory (else zero fill: Dirichlet ghost / padding group)
    bool core[GPT];      // group belongs to the tile's own cells and lies inside the domain
#pragma unroll
    for (int j = 0; j < GPT; ++j) {
        const int g = tid + j * NT;
        const bool act = g < G;
        const int r = g / WQ, q = g % WQ;
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
    // Byte offsets inside one entry fit 32 bits (the launcher checks cells * sizeof(real) < 4 GiB).
    const char* const bR = reinterpret_cast<const char*>(gR);
    const char* const bI = reinterpret_cast<const char*>(gI);
    const char* const bV = reinterpret_cast<const char*>(gV);
    const unsigned plane_bytes = (unsigned)plane * (unsigned)sizeof(real);
    int pz_next;                                     // wrapped index of the next plane to stage
    {
        bool ok_unused;
        pz_next = (P.bcz == BC_PERIODIC) ? zplane(Z0 - H, ok_unused) : Z0 - H;
    }
    auto issue_plane = [&](int slot_idx) {           // stage the next plane of the march into ring slot slot_idx
        const bool zok = (P.bcz == BC_PERIODIC) || (pz_next >= 0 && pz_next < P.nz);
        const unsigned pb = zok ? (unsigned)pz_next * plane_bytes : 0u;
        real* dst = ringR + slot_idx * PS + soff0;
#pragma unroll
        for (int j = 0; j < GPT; ++j) {
            const int nbytes = (ldok[j] && zok) ? 16 : 0;      // 0: zero fill (ghost cells, padding groups)
            const unsigned o = pb + (unsigned)goff[j] * (unsigned)sizeof(real);
            cp_async_16(dst + j * NT * VW, bR + o, nbytes);
            cp_async_16(dst + RD * PS + j * NT * VW, bI + o, nbytes);
            cp_async_16(dst + 2 * RD * PS + j * NT * VW, bV + o, nbytes);
        }
        ++pz_next;
        if (P.bcz == BC_PERIODIC && pz_next == P.nz) pz_next = 0;
    };

    const int niter = bzc + 2 * H;                   // planes Z0-H .. Z0+bzc+H-1 enter the pipeline

    // mask of planes Z0-H-1 .. Z0+bzc+H-1 (0 outside a Dirichlet domain: forces ghost planes to zero)
    for (int q = tid; q < niter + 1; q += NT) {
        bool zok;
        const int pz = zplane(Z0 - H - 1 + q, zok);
        smask[q] = zok ? gM[pz] : (real)0;
    }
    // exchange planes start defined (they are read one iteration before they are first written)
    for (int q = tid; q < (NS - 1) * XD * PS; q += NT) exch[q] = 0;

    Q qa, qb, qc;
#pragma unroll
    for (int s = 0; s < NS; ++s)
#pragma unroll
        for (int j = 0; j < GPT; ++j)
#pragma unroll
            for (int e = 0; e < VW; ++e) { qa.f[s][j].e[e] = 0; qb.f[s][j].e[e] = 0; qc.f[s][j].e[e] = 0; }
#pragma unroll
    for (int j = 0; j < GPT; ++j)
#pragma unroll
        for (int e = 0; e < VW; ++e) { qa.dg[j].e[e] = 0; qb.dg[j].e[e] = 0; qc.dg[j].e[e] = 0; }
    real mq[NS + 1];
#pragma unroll
    for (int s = 0; s <= NS; ++s) mq[s] = 0;

    // ---- prologue: PF planes in flight -----------------------------------------------------------
#pragma unroll
    for (int t = 0; t < PF; ++t) { if (t < niter) issue_plane(t % RD); cp_async_commit(); }

    // One iteration of the march: plane p = Z0-H+t has arrived.  `old`/`mid` hold planes p-s-2 / p-s-1 of
    // every stage s; `nw` receives plane p-s.  (old, mid, nw) rotate by renaming: see the calls below.
    // `ph` = t % 3 is a compile-time constant of the unrolled march, so every shared-memory offset below is
    // an immediate relative to one per-thread base register.
    auto body = [&](const int t, auto phase, Q& old, Q& mid, Q& nw) {
        constexpr int ph = decltype(phase)::value;
        constexpr int ph_prev = (ph + 2) % 3;
        cp_async_wait<PF - 1>();
        __syncthreads();
        if (t + PF < niter) issue_plane((ph + PF) % RD);
        cp_async_commit();

        const int p = Z0 - H + t;
        const real* curR = ringR + ph * PS + soff0;
        constexpr int prvo_c = ph_prev * PS;
        const int prvo = prvo_c + soff0;
#pragma unroll
        for (int s = NS; s > 1; --s) mq[s] = mq[s - 1];
        mq[1] = smask[t];                            // plane p-1

#pragma unroll
        for (int j = 0; j < GPT; ++j) {
            const int jo = j * NT * VW;
            V4 dg_oldest;
            if (NS > 3) dg_oldest = nw.dg[j];        // created three iterations ago: plane p-4
            nw.f[0][j] = *reinterpret_cast<const V4*>(curR + jo);
            const V4 iold = *reinterpret_cast<const V4*>(ringI + prvo + jo);
            const V4 vraw = *reinterpret_cast<const V4*>(ringV + prvo + jo);
#pragma unroll
            for (int e = 0; e < VW; ++e) nw.dg[j].e[e] = fma(cv, vraw.e[e], c6);

#pragma unroll
            for (int s = 1; s <= NS; ++s) {
                const V4& ctr = mid.f[s - 1][j];
                const V4& zlo = old.f[s - 1][j];
                const V4& zhi = nw.f[s - 1][j];
                const V4& older = (s == 1) ? iold : old.f[s >= 2 ? s - 2 : 0][j];
                const V4& dg = (s == 1) ? nw.dg[j] : (s == 2) ? mid.dg[j] : (s == 3) ? old.dg[j] : dg_oldest;
                // plane holding the centre values of this stage (written during the previous iteration)
                const real* cplane = ((s == 1) ? (ringR + prvo) : (exch + ((s >= 2 ? s - 2 : 0) * XD + ph_prev) * PS + soff0)) + jo;
                // x neighbours: shuffles inside the warp; the two warp-edge lanes take theirs from shared memory
                // with ONE load per warp (lane 31 reads its right neighbour, all others lane 0's left neighbour)
                const real edge = cplane[edge_off];
                const real xm_s = __shfl_up_sync(0xffffffffu, ctr.e[VW - 1], 1);
                const real xp_s = __shfl_down_sync(0xffffffffu, ctr.e[0], 1);
                const real xm = (lane == 0) ? edge : xm_s;
                const real xp = (lane == 31) ? edge : xp_s;
                const V4 ym = *reinterpret_cast<const V4*>(cplane - WQ * VW);
                const V4 yp = *reinterpret_cast<const V4*>(cplane + WQ * VW);
                const real m = ldok[j] ? mq[s] : (real)0;
                V4 out;
#pragma unroll
                for (int e = 0; e < VW; ++e) {
                    const real left = (e == 0) ? xm : ctr.e[e - 1];
                    const real right = (e == VW - 1) ? xp : ctr.e[e + 1];
                    const real nb = ((left + right) + (ym.e[e] + yp.e[e])) + (zlo.e[e] + zhi.e[e]);
                    const real upd = fma(c, nb, -dg.e[e] * ctr.e[e]);
                    out.e[e] = m * ((s & 1) ? older.e[e] + upd : older.e[e] - upd);
                }
                if (s < NS) {
                    nw.f[s][j] = out;
                    *reinterpret_cast<V4*>(exch + ((s - 1) * XD + ph) * PS + soff0 + jo) = out;
                }
                if (s == NS - 1) {                   // I^{n+T-1/2} at plane p-NS+1
                    const int pz = p - (NS - 1);
                    if (core[j] && pz >= Z0 && pz < Z0 + bzc)
                        *reinterpret_cast<V4*>(oI + (long long)pz * plane + goff[j]) = out;
                }
                if (s == NS) {                       // R^{n+T} at plane p-NS
                    const int pz = p - NS;
                    if (core[j] && pz >= Z0 && pz < Z0 + bzc)
                        *reinterpret_cast<V4*>(oR + (long long)pz * plane + goff[j]) = out;
                }
            }
        }
    };

#pragma unroll 1
    for (int t = 0; t < niter; t += 3) {
        body(t, std::integral_constant<int, 0>{}, qa, qb, qc);
        if (t + 1 >= niter) break;
        body(t + 1, std::integral_constant<int, 1>{}, qb, qc, qa);
        if (t + 2 >= niter) break;
        body(t + 2, std::integral_constant<int, 2>{}, qc, qa, qb);
    }
    cp_async_wait<0>();
}

}  // namespace tdse
