// tdse_kernels_fused.cuh -- the fused, temporally blocked FDTD step for sm_100a.
//
// One launch advances every batch entry by T full time steps = 2T half-steps ("stages"):
//   stage 2m+1: I^{n+m+1/2} = M[k] * ( I^{n+m-1/2} + lap_c(R^{n+m})     - (2(cx+cy+cz) + c_v V) R^{n+m}     )   eq (9)
//   stage 2m+2: R^{n+m+1}   = M[k] * ( R^{n+m}     - lap_c(I^{n+m+1/2}) + (2(cx+cy+cz) + c_v V) I^{n+m+1/2} )   eq (8)
// where lap_c(f) = cx (f_{i+1} + f_{i-1}) + cy (f_{j+1} + f_{j-1}) + cz (f_{k+1} + f_{k-1}) (the -2 f of each second
// difference is folded into the diagonal), boundary handling per eqs (13)-(14) PAPER.md:126-136 (periodic) or zero-Dirichlet, and the
// absorbing mask M[k] (eq (10) PAPER.md:89-94 as a polynomial mask) fused into the same pass.
//
// Design (differs from the paper's one-thread-per-point kernel, on purpose):
//   * a CTA owns an xy tile (BX x BY cells + halo of 2T) of one batch entry and marches a z chunk;
//     ping-pong buffers (Rin,Iin -> Rout,Iout) make neighbouring tiles independent;
//   * planes of R, I, V (tile + halo) arrive in a shared-memory ring through TMA (cp.async.bulk.tensor, one
//     elected thread, mbarrier completion, PF planes ahead).  Device storage carries a frame of periodic
//     images / Dirichlet zeros around every xy plane (tdse_common.cuh), so a box never wraps in x or y;
//     out-of-range z planes (Dirichlet ghosts) are zero-filled by the TMA unit, periodic z wraps the plane
//     index.  The 5-d tensor view (x, row pair, row parity, z, entry) makes one box land as two
//     half-planes (even rows, odd rows) so that every 16-byte shared-memory access of a warp is contiguous;
//   * a thread owns a 2-row x 16-byte patch of the tile (rows 2rp, 2rp+1).  Per stage it keeps the previous
//     two z-planes of its cells in registers (register-rotated z neighbours: the march is unrolled by 3 so
//     the rotation costs no moves); the y neighbour between its two rows is a register, the outer two y
//     neighbours come from the stage's shared-memory exchange plane, x neighbours from warp shuffles (the
//     two warp-edge lanes read shared memory);
//   * all 2T stages of the software pipeline run between two __syncthreads(); stage s works on plane p-s
//     while planes p+1 .. p+PF are in flight;
//   * cells of the tile next to a periodic face are stored twice (corner cells four times): once in place and
//     once as the image inside the frame, which is what the neighbouring tile's box reads in the next launch;
//   * halo cells are recomputed, not exchanged: the region shrinks by one cell per stage, and values
//     outside that shrinking region are garbage that never reaches a cell that is stored.
// Compulsory HBM traffic: 5 words per cell per launch, i.e. 5/T words per cell-update.
#pragma once
#include <cuda.h>

#include <type_traits>

#include "tdse_common.cuh"

namespace tdse {

struct FusedParams {
    const void* Rin; const void* Iin; const void* V;   // [batch][nz][ny][nx]
    void* Rout; void* Iout;
    const void* mask;                                  // real[nz]
    int nx, ny, nz, batch;
    int bcx, bcy, bcz;
    int px, py;                                        // framed row length / rows per plane
    int tiles_x, tiles_y, nchunks, bz;                 // z chunk length (last chunk may be shorter)
    double cx, cy, cz, cv;                             // PAPER.md:87 (one coefficient per axis)
    float cxf, cyf, czf, cvf, c2f;                     // the same and 2(cx+cy+cz), rounded once on the host for float contexts
    unsigned long long entry_bytes;                    // px*py*nz*sizeof(real)
};

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];\n" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// one box (W x NP x 2 x 1 x 1) of the 5-d view (x, row pair, row parity, z, entry): lands as [parity][pair][x]
__device__ __forceinline__ void tma_load_5d(void* smem_dst, const CUtensorMap* map, unsigned long long* bar,
                                            int c0, int c1, int c2, int c3, int c4)
{
    asm volatile(
        "cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];\n"
        ::"r"(smem_u32(smem_dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4) : "memory");
}

// 16-byte global store under a predicate (no branch)
__device__ __forceinline__ void st_global_pred(void* p, const Pack<float>& v, int pred)
{
    asm volatile("{\n.reg .pred q;\nsetp.ne.s32 q, %5, 0;\n@q st.global.v4.f32 [%0], {%1, %2, %3, %4};\n}\n"
                 ::"l"(p), "f"(v.e[0]), "f"(v.e[1]), "f"(v.e[2]), "f"(v.e[3]), "r"(pred) : "memory");
}
__device__ __forceinline__ void st_global_pred(void* p, const Pack<double>& v, int pred)
{
    asm volatile("{\n.reg .pred q;\nsetp.ne.s32 q, %3, 0;\n@q st.global.v2.f64 [%0], {%1, %2};\n}\n"
                 ::"l"(p), "d"(v.e[0]), "d"(v.e[1]), "r"(pred) : "memory");
}

template <typename real, int T_, int BX_, int BY_, int NT_, int PF_>
struct FusedTraits {
    static constexpr int T = T_, BX = BX_, BY = BY_, NT = NT_, PF = PF_;
    static constexpr int VW = 16 / sizeof(real);
    static constexpr int NS = 2 * T;                           // stages per launch
    static constexpr int H = 2 * T;                            // halo (cells) in y, planes in z
    static constexpr int HX = ((2 * T + VW - 1) / VW) * VW;    // halo in x, vector aligned
    static constexpr int W = BX + 2 * HX;                      // row length of the staged tile
    static constexpr int RH = BY + 2 * H;                      // rows of the staged tile
    static constexpr int WQ = W / VW;                          // 16-byte groups per row
    static constexpr int NP = RH / 2;                          // row pairs
    static constexpr int G2 = WQ * NP;                         // thread slots (one per row pair x group)
    static constexpr int A128 = 128 / sizeof(real);            // elements per 128 bytes (TMA destination alignment)
    static constexpr int HP = NP * W;                          // half-plane stride: even rows, then odd rows (one dense TMA box)
    static constexpr int PS = 2 * HP;                          // plane stride in shared memory (elements)
    static constexpr int GUARD = ((W + A128 - 1) / A128) * A128;     // >= one row before the first / after the last plane
    static constexpr unsigned BOX_BYTES = (unsigned)(PS * sizeof(real));        // bytes one box (W x NP x 2) delivers
    static_assert((PS * sizeof(real)) % 128 == 0, "ring slots must stay 128-byte aligned for TMA");
    static constexpr int RD = PF + 2;                          // ring depth (planes p+PF .. p+1 in flight, p, p-1)
    static constexpr int XD = 2;                               // exchange planes per stage (written at t, read at t+1)
    static constexpr int NPLANES = 3 * RD + (NS - 1) * XD;
    static constexpr size_t SMEM_FIXED = ((size_t)NPLANES * PS + 2 * GUARD) * sizeof(real) + 128 /*alignment slack*/ + 64 /*mbarriers*/;
    // + (bz + 2H + 2) mask values, added by the launcher
    static_assert(RD <= 7, "mbarrier block holds 8 barriers: RD ring slots + the iteration barrier of the SPLIT variant");
    static_assert(H <= PADY && HX <= PADX, "the storage frame must cover the halo");
    static_assert(BX % VW == 0, "tile width must be a multiple of the vector width");
    static_assert(RH % 2 == 0, "rows are owned in pairs");
    static_assert(NT % 32 == 0, "whole warps");
    static_assert(NT >= G2, "one thread per row pair and group");
    static_assert(T == 1 || T == 2, "queue rotation below is written for T = 1, 2");
};

template <typename real, int NS>
struct Queue {                       // one z-plane worth of per-thread pipeline state (rows lo = 0, hi = 1)
    Pack<real> f[NS][2];             // f[s]: field after stage s (s = 0: R as loaded)
    Pack<real> dg[2];                // 6c + c_v V of the plane that entered together with f[0]
};

// GHOSTXY: x or y is a Dirichlet axis, so a tile may hold ghost cells that must stay zero (per-thread mask).
// MINB: CTAs that must fit on one SM (small tiles run several independent CTAs per SM).
// SPLIT: the block barrier per plane becomes an mbarrier that a warp arrives at once its shared-memory traffic of
// the iteration is done and waits for only when it needs the others' exchange planes in the next iteration; the work in
// between (global stores, the wait for the next plane, the ring loads and all of stage 1, which needs no exchange
// plane) absorbs the skew between warps instead of idling at a barrier.  Same arithmetic, same order: bit-identical.
// Worth 2-5 % where a launch is one wave of short chunks (64^3, one 128^3 f64 grid), nothing on the multi-wave grids.
template <typename real, int T, int BX, int BY, int NT, int PF, bool GHOSTXY, int MINB = 1, bool SPLIT = false>
__global__ void __launch_bounds__(NT, MINB)
fdtd_fused_kernel(const FusedParams P, const __grid_constant__ CUtensorMap tmR,
                  const __grid_constant__ CUtensorMap tmI, const __grid_constant__ CUtensorMap tmV)
{
    using Tr = FusedTraits<real, T, BX, BY, NT, PF>;
    using V4 = Pack<real>;
    using Q = Queue<real, Tr::NS>;
    constexpr int VW = Tr::VW, NS = Tr::NS, H = Tr::H, HX = Tr::HX, WQ = Tr::WQ, W = Tr::W;
    constexpr int G2 = Tr::G2, PS = Tr::PS, HP = Tr::HP, RD = Tr::RD, XD = Tr::XD;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    unsigned char* const smem_al = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);   // TMA wants 128-byte aligned boxes
    real* const ringR = reinterpret_cast<real*>(smem_al) + Tr::GUARD;
    real* const ringI = ringR + RD * PS;
    real* const ringV = ringI + RD * PS;
    real* const exch = ringV + RD * PS;                    // stage s output of iteration t at exch[((s-1)*XD + t%2) * PS]
    unsigned long long* const full = reinterpret_cast<unsigned long long*>(exch + (NS - 1) * XD * PS + Tr::GUARD);   // full[slot]: plane landed
    unsigned long long* const iter_done = full + 7;        // SPLIT: one arrival per warp and iteration
    real* const smask = reinterpret_cast<real*>(full + 8); // smask[q] = mask of plane Z0-H-1+q

    const int tid = threadIdx.x, lane = tid & 31;
    const int ntiles = P.tiles_x * P.tiles_y;
    int bid = blockIdx.x;
    const int tile = bid % ntiles; bid /= ntiles;
    const int chunk = bid % P.nchunks;
    const int b = bid / P.nchunks;
    const int X0 = (tile % P.tiles_x) * BX, Y0 = (tile / P.tiles_x) * BY;
    const int Z0 = chunk * P.bz;
    const int bzc = min(P.bz, P.nz - Z0);
    const real* __restrict__ gM = static_cast<const real*>(P.mask);
    real cx, cy, cz, cv, c2;                        // c2 = 2 (cx + cy + cz): the diagonal of the three second differences
    if constexpr (std::is_same<real, float>::value) { cx = P.cxf; cy = P.cyf; cz = P.czf; cv = P.cvf; c2 = P.c2f; }
    else { cx = P.cx; cy = P.cy; cz = P.cz; cv = P.cv; c2 = 2.0 * (P.cx + P.cy + P.cz); }

    // ---- per-thread geometry, fixed for the whole march ---------------------------------------
    // Threads beyond the last slot repeat the last slot (a halo corner): same loads, same values, no stores.
    const int slot = min(tid, G2 - 1);
    const int rp = slot / WQ, q = slot % WQ;
    const int soff = rp * W + q * VW;                // even-row group inside a plane; odd row at soff + HP
    // x neighbours across the warp edge: lane 31 reads the element right of its group, every other lane the
    // element left of lane 0's group (one broadcast address) -- only lanes 0 and 31 use what they read.
    const int soff_lane0 = __shfl_sync(0xffffffffu, soff, 0);
    const int edge_off = (lane == 31) ? VW : (soff_lane0 - 1 - soff);

    unsigned goff[2];    // byte offset of the group inside a framed plane
    int inside[2];       // group lies inside the domain (else: Dirichlet ghost, must stay zero)
    int core[2];         // group belongs to the tile's own cells and lies inside the domain
    int img_x = 0, img_y[2] = {0, 0};   // byte shifts of the periodic images this thread also stores (0: none)
    {
        const int xg = X0 - HX + q * VW;
        const bool inx = P.bcx == BC_PERIODIC || (xg >= 0 && xg < P.nx);
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const int r = 2 * rp + j;
            const int yg = Y0 - H + r;
            const bool iny = P.bcy == BC_PERIODIC || (yg >= 0 && yg < P.ny);
            inside[j] = inx && iny;
            goff[j] = (unsigned)((yg + PADY) * P.px + xg + PADX) * (unsigned)sizeof(real);
            core[j] = tid < G2 && q * VW >= HX && q * VW < HX + BX && r >= H && r < H + BY &&
                      xg < P.nx && yg < P.ny;   // xg, yg >= 0 is implied for core groups
            if (core[j] && P.bcy == BC_PERIODIC) {
                if (yg < PADY) img_y[j] = P.ny * P.px * (int)sizeof(real);
                else if (yg >= P.ny - PADY) img_y[j] = -P.ny * P.px * (int)sizeof(real);
            }
        }
        if ((core[0] || core[1]) && P.bcx == BC_PERIODIC) {
            if (xg < PADX) img_x = P.nx * (int)sizeof(real);
            else if (xg >= P.nx - PADX) img_x = -P.nx * (int)sizeof(real);
        }
    }
    const bool warp_img_x = __any_sync(0xffffffffu, img_x != 0);                 // warp-uniform: no divergence
    const bool warp_img_y = __any_sync(0xffffffffu, (img_y[0] | img_y[1]) != 0);

    // Byte offsets inside one entry fit 32 bits (the launcher checks pcells * sizeof(real) < 4 GiB).
    const unsigned long long ebase = (unsigned long long)b * P.entry_bytes;
    char* const oR = static_cast<char*>(P.Rout) + ebase;
    char* const oI = static_cast<char*>(P.Iout) + ebase;
    const unsigned plane_bytes = (unsigned)(P.px * P.py) * (unsigned)sizeof(real);

    // ---- TMA producer (thread 0): plane pz_next -> ring slot, two half-plane boxes per array ---------
    int pz_next = Z0 - H;                            // next plane to stage (wrapped when z is periodic)
    if (P.bcz == BC_PERIODIC) pz_next = wrap_index(pz_next, P.nz);
    const int box_x = X0 - HX + PADX, box_yp = (Y0 - H + PADY) / 2;   // box origin: x, row pair (Y0-H+PADY is even)
    auto issue_plane = [&](int ring_off, int slot_idx) {
        // a Dirichlet ghost plane has an out-of-range z coordinate: the TMA unit fills the box with zeros
        unsigned long long* bar = full + slot_idx;
        mbar_expect_tx(bar, 3u * Tr::BOX_BYTES);
        real* dst = ringR + ring_off;
        tma_load_5d(dst, &tmR, bar, box_x, box_yp, 0, pz_next, b);
        tma_load_5d(dst + RD * PS, &tmI, bar, box_x, box_yp, 0, pz_next, b);
        tma_load_5d(dst + 2 * RD * PS, &tmV, bar, box_x, box_yp, 0, pz_next, b);
        ++pz_next;
        if (P.bcz == BC_PERIODIC && pz_next == P.nz) pz_next = 0;
    };

    const int niter = bzc + 2 * H;                   // planes Z0-H .. Z0+bzc+H-1 enter the pipeline

    // mask of planes Z0-H-1 .. Z0+bzc+H-1 (0 outside a Dirichlet domain: forces ghost planes to zero)
    for (int i = tid; i < niter + 1; i += NT) {
        int pz = Z0 - H - 1 + i;
        bool zok = pz >= 0 && pz < P.nz;
        if (P.bcz == BC_PERIODIC) { pz = wrap_index(pz, P.nz); zok = true; }
        smask[i] = zok ? gM[pz] : (real)0;
    }
    // exchange planes start defined (they are read one iteration before they are first written)
    for (int i = tid; i < (NS - 1) * XD * PS; i += NT) exch[i] = 0;

    Q qa, qb, qc;
#pragma unroll
    for (int s = 0; s < NS; ++s)
#pragma unroll
        for (int j = 0; j < 2; ++j)
#pragma unroll
            for (int e = 0; e < VW; ++e) { qa.f[s][j].e[e] = 0; qb.f[s][j].e[e] = 0; qc.f[s][j].e[e] = 0; }
#pragma unroll
    for (int j = 0; j < 2; ++j)
#pragma unroll
        for (int e = 0; e < VW; ++e) { qa.dg[j].e[e] = 0; qb.dg[j].e[e] = 0; qc.dg[j].e[e] = 0; }
    real mq[NS + 1];
#pragma unroll
    for (int s = 0; s <= NS; ++s) mq[s] = 0;

    // ---- prologue: barriers, PF planes in flight --------------------------------------------------
    if (tid == 0) {
#pragma unroll
        for (int i = 0; i < RD; ++i) mbar_init(full + i, 1);
        if (SPLIT) mbar_init(iter_done, NT / 32);
        asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
    }
    // Programmatic dependent launch: everything above touched only shared memory, kernel parameters and the mask
    // table (which no kernel writes).  The previous launch in the stream wrote the arrays this one reads and
    // read the arrays this one writes, so every thread waits for it to complete before its first global
    // access; only then may the launch after this one become resident (at most one launch runs ahead).
    asm volatile("griddepcontrol.wait;\n" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory");
    if (tid == 0) {
#pragma unroll
        for (int t = 0; t < PF; ++t) if (t < niter) issue_plane(t * PS, t);
    }
    __syncthreads();                                 // barriers initialised before anyone waits on them
    // ring slot offsets (elements) of plane p (cur), p-1 (prev) and of the slot plane p+PF goes to (fill);
    // exchange-plane offsets written this iteration (xw) and read from the previous one (xr)
    auto ring_next = [](int o) { return (o + PS == RD * PS) ? 0 : o + PS; };
    int ro_cur = 0, ro_prev = (RD - 1) * PS, ro_fill = (PF % RD) * PS;
    int sl_cur = 0, sl_fill = PF % RD;               // the same as slot indices (barrier array)
    unsigned par = 0;                                // phase parity of full[sl_cur]
    unsigned dpar = 0;                               // SPLIT: phase parity of iter_done
    int xw = 0, xr = PS;

    // Address of the thread's upper row in plane p-NS of R-out, advanced by one plane per iteration (while p-NS < Z0 it points
    // below the chunk and is not dereferenced).  Everything a thread stores sits at a uniform or per-thread constant distance
    // from it -- lower row, I-out one plane further, periodic images -- so a store costs one 64-bit add instead of an
    // offset multiply-add chain (the stores and their address arithmetic are 16 % of the instruction stream).
    char* out_r = oR + (long long)(Z0 - H - NS) * (long long)plane_bytes + goff[0];
    const long long i_from_r = (oI - oR) + (long long)plane_bytes;   // I-out plane p-NS+1 relative to R-out plane p-NS
    const unsigned row_bytes = goff[1] - goff[0];

    // one of the thread's two rows (j) of a finished plane -> global memory, plus its periodic images inside the frame;
    // d0 = address of the thread's upper row in that plane
    auto store_row = [&](char* d0, const V4& v, const int j) {
        // predicated 16-byte stores, no divergent branches (a branch region per row and image cost more than the
        // stores themselves: profiles/README.md); only warps that hold a y-face row enter the y-image part
        char* const d = j ? d0 + row_bytes : d0;
        st_global_pred(d, v, core[j]);
        if (warp_img_x) st_global_pred(d + img_x, v, core[j] && img_x);
        if (warp_img_y) {
            st_global_pred(d + img_y[j], v, img_y[j]);
            st_global_pred(d + img_y[j] + img_x, v, img_y[j] && img_x);
        }
    };
    auto store_rows = [&](char* d0, const V4 (&out)[2]) { store_row(d0, out[0], 0); store_row(d0, out[1], 1); };

    // One iteration of the march: plane p = Z0-H+t has arrived.  `old`/`mid` hold planes p-s-2 / p-s-1 of
    // every stage s; `nw` receives plane p-s.  (old, mid, nw) rotate by renaming: see the calls below.
    auto body = [&](const int t, Q& old, Q& mid, Q& nw) {
        mbar_wait(full + sl_cur, par);               // plane p has landed (issued PF iterations ago)
        if (!SPLIT) {
            __syncthreads();                         // everyone is done with iteration t-1 (ring slot p-2, exchange planes)
            // refill the slot of plane p-2: its last readers passed the barrier above (reads ordered before the async write)
            if (tid == 0 && t + PF < niter) issue_plane(ro_fill, sl_fill);
        }

        const int p = Z0 - H + t;
#pragma unroll
        for (int s = NS; s > 1; --s) mq[s] = mq[s - 1];
        mq[1] = smask[t];                            // plane p-1

        V4 dg_oldest[2];
        V4 iold[2];
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            if (NS > 3) dg_oldest[j] = nw.dg[j];     // created three iterations ago: plane p-4
            nw.f[0][j] = *reinterpret_cast<const V4*>(ringR + ro_cur + soff + j * HP);
            iold[j] = *reinterpret_cast<const V4*>(ringI + ro_prev + soff + j * HP);
            const V4 vraw = *reinterpret_cast<const V4*>(ringV + ro_prev + soff + j * HP);
#pragma unroll
            for (int e = 0; e < VW; ++e) nw.dg[j].e[e] = fma(cv, vraw.e[e], c2);
        }

#pragma unroll
        for (int s = 1; s <= NS; ++s) {
            if (SPLIT && s == 2) {
                // Stage 1 above read the ring only.  From here on the iteration reads the exchange planes the others wrote
                // in iteration t-1 and overwrites the ones they read then: wait until every warp has arrived for t-1.
                if (t > 0) { mbar_wait(iter_done, dpar); dpar ^= 1u; }
                // the same arrivals say that the ring slot of plane p-2 has been read for the last time: refill it
                if (tid == 0 && t + PF < niter) issue_plane(ro_fill, sl_fill);
#pragma unroll
                for (int j = 0; j < 2; ++j) *reinterpret_cast<V4*>(exch + xw + soff + j * HP) = nw.f[1][j];
            }
            // plane holding the centre values of this stage (written during the previous iteration)
            const real* cplane = ((s == 1) ? (ringR + ro_prev) : (exch + (s >= 2 ? s - 2 : 0) * XD * PS + xr)) + soff;
            const V4 ym = *reinterpret_cast<const V4*>(cplane + HP - W);     // row 2rp-1: odd row of pair rp-1
            const V4 yp = *reinterpret_cast<const V4*>(cplane + W);          // row 2rp+2: even row of pair rp+1
            real edge[2];
            edge[0] = cplane[edge_off];
            edge[1] = cplane[HP + edge_off];
            V4 out[2];
#pragma unroll
            for (int j = 0; j < 2; ++j) {
                const V4& ctr = mid.f[s - 1][j];
                const V4& zlo = old.f[s - 1][j];
                const V4& zhi = nw.f[s - 1][j];
                const V4& older = (s == 1) ? iold[j] : old.f[s >= 2 ? s - 2 : 0][j];
                const V4& dg = (s == 1) ? nw.dg[j] : (s == 2) ? mid.dg[j] : (s == 3) ? old.dg[j] : dg_oldest[j];
                const V4& ylo = (j == 0) ? ym : mid.f[s - 1][0];
                const V4& yhi = (j == 0) ? mid.f[s - 1][1] : yp;
                const real xm_s = __shfl_up_sync(0xffffffffu, ctr.e[VW - 1], 1);
                const real xp_s = __shfl_down_sync(0xffffffffu, ctr.e[0], 1);
                const real xm = (lane == 0) ? edge[j] : xm_s;
                const real xp = (lane == 31) ? edge[j] : xp_s;
                const real m = (GHOSTXY && !inside[j]) ? (real)0 : mq[s];
#pragma unroll
                for (int e = 0; e < VW; ++e) {
                    const real left = (e == 0) ? xm : ctr.e[e - 1];
                    const real right = (e == VW - 1) ? xp : ctr.e[e + 1];
                    const real xs = left + right, ys = ylo.e[e] + yhi.e[e], zs = zlo.e[e] + zhi.e[e];
                    // odd stages: older + (cx xs + cy ys + cz zs - dg ctr); even stages: older - (...).  zs (which needs
                    // this iteration's output of the previous stage) enters the chain last.
                    const real u = (s & 1) ? fma(cz, zs, fma(-dg.e[e], ctr.e[e], fma(cy, ys, fma(cx, xs, older.e[e]))))
                                           : fma(-cz, zs, fma(dg.e[e], ctr.e[e], fma(-cy, ys, fma(-cx, xs, older.e[e]))));
                    out[j].e[e] = m * u;
                }
            }
            if (s < NS) {
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    nw.f[s][j] = out[j];
                    if (!(SPLIT && s == 1)) *reinterpret_cast<V4*>(exch + (s - 1) * XD * PS + xw + soff + j * HP) = out[j];
                }
            }
            // I^{n+T-1/2} of the PREVIOUS iteration (plane p-NS, the same plane index as this iteration's R-out) sits in the
            // queue anyway: its two rows are stored here, spread over the stages, instead of right behind stage NS-1, so that
            // the global stores of an iteration do not all leave in one burst at its end (measured: +3 to +7 % on the f32
            // grids, profiles/r02_experiments.md).  The last iteration produces no valid I plane: nothing is left over.
            constexpr int I0_AT = NS == 2 ? 1 : (sizeof(real) == 4 ? 2 : 1), I1_AT = NS == 2 ? 2 : 3;
            if (!SPLIT && (s == I0_AT || s == I1_AT)) {
                const int pz = p - NS;
                if (pz >= Z0 && pz < Z0 + bzc) {
                    char* const d = out_r + (i_from_r - (long long)plane_bytes);
                    if (s == I0_AT) store_row(d, mid.f[NS - 1][0], 0);
                    if (s == I1_AT) store_row(d, mid.f[NS - 1][1], 1);
                }
            }
            if (s == NS) {                           // R^{n+T} at plane p-NS
                if (SPLIT) {
                    // this warp's shared-memory traffic of iteration t is done: arrive, then store (I from the queue)
                    __syncwarp();
                    if (lane == 0) mbar_arrive(iter_done);
                    const int pzi = p - (NS - 1);
                    if (pzi >= Z0 && pzi < Z0 + bzc) store_rows(out_r + i_from_r, nw.f[NS - 1]);
                }
                const int pz = p - NS;
                if (pz >= Z0 && pz < Z0 + bzc) store_rows(out_r, out);
            }
        }
        out_r += plane_bytes;
        ro_prev = ro_cur; ro_cur = ring_next(ro_cur); ro_fill = ring_next(ro_fill);
        if (++sl_cur == RD) { sl_cur = 0; par ^= 1u; }
        if (++sl_fill == RD) sl_fill = 0;
        xr = xw; xw = PS - xw;
    };

#pragma unroll 1
    for (int t = 0; t < niter; t += 3) {
        body(t, qa, qb, qc);
        if (t + 1 >= niter) break;
        body(t + 1, qb, qc, qa);
        if (t + 2 >= niter) break;
        body(t + 2, qc, qa, qb);
    }
}

}  // namespace tdse
