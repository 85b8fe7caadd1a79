// tdse.cu -- C-ABI of libtdse (include/tdse.h): context, host-side scheduling, kernel launches.
// sm_100a only.  No CPU fallback: every entry point fails with TDSE_ECUDA without a device.
#include "../../include/tdse.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <limits>
#include <map>
#include <new>
#include <string>
#include <vector>

#include "tdse_common.cuh"
#include "tdse_kernels_basic.cuh"
#include "tdse_kernels_fused.cuh"

using namespace tdse;

namespace {

thread_local std::string g_create_error;    // the context-free error slot (tdse_last_error(NULL)): one per host thread

constexpr size_t kAlign = 256;
constexpr int kMaxDevices = 64;
inline size_t align_up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

}  // namespace

struct tdse_ctx {
    Grid g{};
    int dtype = TDSE_F64;
    size_t w = 8;                       // bytes per element
    double dx = 0, dt = 0, mass = 0, hbar = 0;
    Mesh m{};                           // spacings (dx, dy, dz) and coefficients cx, cy, cz, c_v of PAPER.md:87
    int absorb_lo = 0, absorb_hi = 0, power = 2;
    double strength = 0.0;

    // workspace
    void* ws = nullptr;
    size_t ws_bytes = 0;
    bool ws_owned = false;
    bool pingpong = false;
    size_t arr_bytes = 0;               // aligned bytes of one [batch][nz][ny][nx] array
    void* R[2] = {nullptr, nullptr};
    void* I[2] = {nullptr, nullptr};
    void* V = nullptr;
    int cur = 0;
    cudaStream_t stream = nullptr;
    int device = 0;                     // the device that was current in tdse_create: every later call runs there

    // small library-owned buffers
    void* mask_dev = nullptr;           // real[nz]
    std::vector<double> mask_host;
    double* D = nullptr;                // [batch][ny][nx]
    double* trace = nullptr;            // [batch][max_samples]
    double* partial = nullptr;          // scratch for reductions
    unsigned* done = nullptr;           // detector kernel: blocks finished per entry (returns to 0 after every sample)
    size_t partial_n = 0;
    double* scalars = nullptr;          // 4 doubles
    AtomRange* pot_ranges = nullptr;    // tdse_set_potential_batch: per-entry slices of the atom array [batch]
    int* pot_count = nullptr;           //   shared-prefix length found on the device
    double* pot_prefix = nullptr;       //   fp64 sums of the shared prefix, flat [nz][ny][nx]
    double* cell_stage = nullptr;       // tdse_set_potential_cell: device copy of a host unit cell
    size_t cell_cap = 0;
    AtomRec* atoms_dev = nullptr;
    AtomRec* atoms_pin = nullptr;
    int atoms_cap = 0;
    cudaEvent_t atoms_ev = nullptr;
    bool atoms_pending = false;

    int k_det = 0, every = 0, max_samples = 0, nsamples = 0;
    double* frames = nullptr;           // frame mode: [batch][max_frames][ny][nx]
    int max_frames = 0, nframes = 0, frames_t0 = 1;
    // streamed frame mode (tdse_set_frame_stream): a device ring of fs_slots sample slots [slot][batch][ny][nx]; every
    // finished slot leaves on a second stream into the caller's host buffer [batch][fs_capacity][ny][nx]
    double* fs_ring = nullptr;
    double* fs_host = nullptr;
    int fs_slots = 0, fs_capacity = 0;
    bool fs_copy2d = true;              // one strided 2-D copy per slot (host pitch within cudaDevAttrMaxPitch), else one copy per entry
    cudaStream_t fs_stream = nullptr;
    std::vector<cudaEvent_t> fs_written, fs_copied;
    std::vector<char> fs_busy;          // fs_copied[slot] has been recorded since the last reset
    long long steps = 0;
    std::vector<char> have_V, have_state;
    double vabs_max = 0.0;

    // options / info
    int opt_kernel = TDSE_KERNEL_AUTO, opt_tblock = 0, allow_unstable = 0, opt_pf = 0, opt_chunks = 0, opt_pdl = 1, opt_variant = 0;
    long long launches = 0;
    int last_kernel = 0, last_tblock = 0, last_tile_x = 0, last_tile_y = 0, last_chunks = 0;
    int num_sms = 148;
    std::map<int, std::vector<CUtensorMap>> tmaps;   // per fused variant: maps of R[0], I[0], V, R[1], I[1]
    std::string err;
};

namespace {

// Every entry point runs on the context's device whatever device the caller has current, and restores the caller's.
// If the switch cannot be made the entry point must not run at all (it would launch on some other device against this
// device's pointers): ok() is false and ENTER_DEVICE returns TDSE_ECUDA.
struct DeviceScope {
    int prev = -1;
    bool switched = false;
    cudaError_t err = cudaSuccess;
    explicit DeviceScope(const tdse_ctx* c)
    {
        if (!c) return;
        if ((err = cudaGetDevice(&prev)) != cudaSuccess) { cudaGetLastError(); prev = -1; return; }
        if (prev != c->device) {
            if ((err = cudaSetDevice(c->device)) != cudaSuccess) { cudaGetLastError(); return; }
            switched = true;
        }
    }
    bool ok() const { return err == cudaSuccess; }
    ~DeviceScope() { if (switched && cudaSetDevice(prev) != cudaSuccess) cudaGetLastError(); }
    DeviceScope(const DeviceScope&) = delete;
    DeviceScope& operator=(const DeviceScope&) = delete;
};

int fail(tdse_ctx* ctx, int code, const std::string& msg)
{
    if (ctx) ctx->err = msg; else g_create_error = msg;
    return code;
}

#define CU_TRY(ctx, expr)                                                                     \
    do {                                                                                      \
        cudaError_t e__ = (expr);                                                             \
        if (e__ != cudaSuccess)                                                               \
            return fail(ctx, TDSE_ECUDA, std::string(#expr) + ": " + cudaGetErrorString(e__)); \
    } while (0)

#define ENTER_DEVICE(ctx)                                                                          \
    DeviceScope on_device_(ctx);                                                                   \
    if (!on_device_.ok())                                                                          \
        return fail(ctx, TDSE_ECUDA, std::string("cannot make the context's device current: ") + cudaGetErrorString(on_device_.err))

#define CU_LAUNCH_CHECK(ctx)                                                                     \
    do {                                                                                         \
        cudaError_t e__ = cudaGetLastError();                                                    \
        if (e__ != cudaSuccess)                                                                  \
            return fail(ctx, TDSE_ECUDA, std::string("kernel launch: ") + cudaGetErrorString(e__)); \
        ctx->launches++;                                                                         \
    } while (0)

inline size_t elem_bytes(int dtype) { return dtype == TDSE_F32 ? 4 : 8; }

void carve(tdse_ctx* c)
{
    char* base = static_cast<char*>(c->ws);
    c->R[0] = base;
    c->I[0] = base + c->arr_bytes;
    c->V = base + 2 * c->arr_bytes;
    if (c->pingpong) {
        c->R[1] = base + 3 * c->arr_bytes;
        c->I[1] = base + 4 * c->arr_bytes;
    } else {
        c->R[1] = c->I[1] = nullptr;
    }
    c->cur = 0;
    c->tmaps.clear();
    std::fill(c->have_V.begin(), c->have_V.end(), 0);
    std::fill(c->have_state.begin(), c->have_state.end(), 0);
    c->vabs_max = 0.0;
}

int ensure_workspace(tdse_ctx* c)
{
    if (c->ws) return TDSE_OK;
    const size_t bytes = 5 * c->arr_bytes;
    void* p = nullptr;
    cudaError_t e = cudaMalloc(&p, bytes);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(c, TDSE_ENOMEM, std::string("cudaMalloc workspace: ") + cudaGetErrorString(e));
    }
    c->ws = p; c->ws_bytes = bytes; c->ws_owned = true; c->pingpong = true;
    carve(c);
    CU_TRY(c, cudaMemsetAsync(c->ws, 0, bytes, c->stream));   // frames of Dirichlet axes stay zero
    return TDSE_OK;
}

int ensure_partial(tdse_ctx* c, size_t n)
{
    if (n <= c->partial_n) return TDSE_OK;
    if (c->partial) { cudaStreamSynchronize(c->stream); cudaFree(c->partial); c->partial = nullptr; c->partial_n = 0; }
    CU_TRY(c, cudaMalloc(&c->partial, n * sizeof(double)));
    c->partial_n = n;
    return TDSE_OK;
}

// Absorbing mask of include/tdse.h (tdse_set_boundary), double on the host, rounded once to dtype.
int upload_mask(tdse_ctx* c)
{
    const int nz = c->g.nz;
    c->mask_host.assign(nz, 1.0);
    for (int k = 0; k < nz; ++k) {
        double xi = 0.0;
        if (c->absorb_lo > 0 && k < c->absorb_lo) xi = double(c->absorb_lo - k) / double(c->absorb_lo);
        if (c->absorb_hi > 0 && k > nz - 1 - c->absorb_hi) xi = double(k - (nz - 1 - c->absorb_hi)) / double(c->absorb_hi);
        if (xi > 0.0) {
            double p = 1.0;
            for (int q = 0; q < c->power; ++q) p *= xi;
            c->mask_host[k] = 1.0 - c->strength * p;
        }
    }
    if (!c->mask_dev) CU_TRY(c, cudaMalloc(&c->mask_dev, (size_t)nz * c->w));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    if (c->dtype == TDSE_F32) {
        std::vector<float> m(nz);
        for (int k = 0; k < nz; ++k) m[k] = (float)c->mask_host[k];
        CU_TRY(c, cudaMemcpy(c->mask_dev, m.data(), (size_t)nz * 4, cudaMemcpyHostToDevice));
    } else {
        CU_TRY(c, cudaMemcpy(c->mask_dev, c->mask_host.data(), (size_t)nz * 8, cudaMemcpyHostToDevice));
    }
    return TDSE_OK;
}

int reset_detector(tdse_ctx* c)
{
    c->steps = 0;
    c->nsamples = 0;
    c->nframes = 0;                      // streamed mode: frame 0 again; copies still in flight stay ordered on fs_stream
    if (c->D) {
        const long long n = (long long)c->g.batch * c->g.plane;
        fill_zero_kernel<<<(unsigned)std::min<long long>((n + 255) / 256, 4096), 256, 0, c->stream>>>(c->D, n);
        CU_LAUNCH_CHECK(c);
    }
    if (c->trace && c->max_samples > 0) {
        const long long n = (long long)c->g.batch * c->max_samples;
        fill_zero_kernel<<<(unsigned)std::min<long long>((n + 255) / 256, 4096), 256, 0, c->stream>>>(c->trace, n);
        CU_LAUNCH_CHECK(c);
    }
    return TDSE_OK;
}

inline char* entry_ptr(const tdse_ctx* c, void* arr, int b) { return static_cast<char*>(arr) + (size_t)b * c->g.pcells * c->w; }

// Copy one entry between a flat [nz][ny][nx] buffer (C-ABI layout) and the framed device storage.
int copy_entry(tdse_ctx* c, void* dev_entry, void* flat, cudaMemcpyKind kind, bool to_device)
{
    cudaMemcpy3DParms p{};
    const cudaPitchedPtr framed = make_cudaPitchedPtr(dev_entry, (size_t)c->g.px * c->w, (size_t)c->g.px * c->w, (size_t)c->g.py);
    const cudaPitchedPtr plain = make_cudaPitchedPtr(flat, (size_t)c->g.nx * c->w, (size_t)c->g.nx * c->w, (size_t)c->g.ny);
    const cudaPos inner = make_cudaPos((size_t)PADX * c->w, (size_t)PADY, 0), origin = make_cudaPos(0, 0, 0);
    if (to_device) { p.srcPtr = plain; p.srcPos = origin; p.dstPtr = framed; p.dstPos = inner; }
    else           { p.srcPtr = framed; p.srcPos = inner; p.dstPtr = plain; p.dstPos = origin; }
    p.extent = make_cudaExtent((size_t)c->g.nx * c->w, (size_t)c->g.ny, (size_t)c->g.nz);
    p.kind = kind;
    CU_TRY(c, cudaMemcpy3DAsync(&p, c->stream));
    return TDSE_OK;
}

int fill_frame(tdse_ctx* c, void* dev_entry)
{
    const unsigned nblk = (unsigned)((c->g.pcells + 255) / 256);
    if (c->dtype == TDSE_F32) frame_fill_kernel<float><<<nblk, 256, 0, c->stream>>>(c->g, static_cast<float*>(dev_entry));
    else frame_fill_kernel<double><<<nblk, 256, 0, c->stream>>>(c->g, static_cast<double*>(dev_entry));
    CU_LAUNCH_CHECK(c);
    return TDSE_OK;
}

bool entry_range(const tdse_ctx* c, int b, int* b0, int* b1)
{
    if (b == -1) { *b0 = 0; *b1 = c->g.batch; return true; }
    if (b < 0 || b >= c->g.batch) return false;
    *b0 = b; *b1 = b + 1;
    return true;
}

// ---------------------------------------------------------------------------------------------
// TMA descriptors for the fused kernel: the 5-d view (x, row pair, row parity, z, entry) of one framed
// array, box = one tile plane (W x NP x 2 x 1 x 1), which lands as [parity][pair][x].  cuTensorMapEncodeTiled is taken from the
// driver through the runtime (no link against libcuda).
// ---------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn()
{
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
        else
            cudaGetLastError();
    }
    return fn;
}

// maps of R[0], I[0], V, R[1], I[1] for boxes of W columns x NP row pairs
int get_tensor_maps(tdse_ctx* c, int W, int NP, const CUtensorMap** out)
{
    const int key = W * 1024 + NP;
    auto it = c->tmaps.find(key);
    if (it == c->tmaps.end()) {
        EncodeTiledFn enc = encode_tiled_fn();
        if (!enc) return fail(c, TDSE_ECUDA, "fused launch: cuTensorMapEncodeTiled is not available from the driver");
        std::vector<CUtensorMap> maps(5);
        void* arrs[5] = {c->R[0], c->I[0], c->V, c->R[1], c->I[1]};
        const cuuint64_t w = c->w, px = (cuuint64_t)c->g.px, py = (cuuint64_t)c->g.py;
        const cuuint64_t dims[5] = {px, py / 2, 2, (cuuint64_t)c->g.nz, (cuuint64_t)c->g.batch};
        const cuuint64_t strides[4] = {2 * px * w, px * w, px * py * w, px * py * (cuuint64_t)c->g.nz * w};
        const cuuint32_t box[5] = {(cuuint32_t)W, (cuuint32_t)NP, 2, 1, 1};
        const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
        for (int a = 0; a < 5; ++a) {
            const CUresult r = enc(&maps[a], c->dtype == TDSE_F32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64,
                                   5, arrs[a], dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                   CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (r != CUDA_SUCCESS) return fail(c, TDSE_ECUDA, "fused launch: cuTensorMapEncodeTiled failed with code " + std::to_string((int)r));
        }
        it = c->tmaps.emplace(key, std::move(maps)).first;
    }
    *out = it->second.data();
    return TDSE_OK;
}

// z chunking of one fused variant: minimise waves * (chunk length + halo planes) on num_sms * ctas_per_sm slots.
// Also used without launching, to compare variants (auto_tblock).  planes_out = planes one CTA marches times waves.
template <typename real, int T, int BX, int BY, int NT, int PF, int MINB = 1>
int plan_fused(tdse_ctx* c, int ctas_per_sm, int* tiles_x, int* tiles_y, int* bz_out, int* nchunks_out, long long* planes_out)
{
    using Tr = FusedTraits<real, T, BX, BY, NT, PF>;
    constexpr size_t kMaxSmem = MINB == 1 ? 227 * 1024 : (228 * 1024) / MINB - 1024;   // per CTA (1 KB reserved each)
    *tiles_x = (c->g.nx + BX - 1) / BX;
    *tiles_y = (c->g.ny + BY - 1) / BY;
    const long long units = (long long)*tiles_x * *tiles_y * c->g.batch;
    const long long slots = (long long)c->num_sms * ctas_per_sm;
    const int H = Tr::H;
    const int max_bz = (int)((kMaxSmem - Tr::SMEM_FIXED) / sizeof(real)) - 2 * H - 2;   // mask table must fit
    int best_n = 0;
    double best_cost = std::numeric_limits<double>::max();
    const int max_chunks = std::max(1, c->g.nz / 2);   // chunks of >= 2 planes; the cost model below weighs the halo planes
    for (int n = 1; n <= std::max(std::max(max_chunks, c->opt_chunks), (c->g.nz + max_bz - 1) / max_bz); ++n) {
        const int bz = (c->g.nz + n - 1) / n;
        if (bz > max_bz) continue;
        if (c->opt_chunks > 0 && n != std::min(c->opt_chunks, c->g.nz)) continue;
        const int n_eff = (c->g.nz + bz - 1) / bz;
        const long long waves = (units * n_eff + slots - 1) / slots;
        const double cost = (double)waves * (bz + 2 * H + 3);   // +3: pipeline fill/launch overhead in plane units
        if (cost < best_cost - 1e-9) { best_cost = cost; best_n = n_eff; }
    }
    if (best_n == 0) return fail(c, TDSE_EINVAL, "fused launch: no feasible z chunking");
    *bz_out = (c->g.nz + best_n - 1) / best_n;
    *nchunks_out = (c->g.nz + *bz_out - 1) / *bz_out;
    if (planes_out) *planes_out = ((units * *nchunks_out + slots - 1) / slots) * (*bz_out + 2 * H);
    return TDSE_OK;
}

// ---------------------------------------------------------------------------------------------
// fused launch table
// ---------------------------------------------------------------------------------------------
template <typename real, int T, int BX, int BY, int NT, int PF, bool GHOSTXY, int MINB = 1, bool SPLIT = false>
int launch_fused_cfg(tdse_ctx* c, FusedParams& P, int ctas_per_sm = MINB)
{
    using Tr = FusedTraits<real, T, BX, BY, NT, PF>;
    auto kern = fdtd_fused_kernel<real, T, BX, BY, NT, PF, GHOSTXY, MINB, SPLIT>;
    constexpr size_t kMaxSmem = MINB == 1 ? 227 * 1024 : (228 * 1024) / MINB - 1024;   // per CTA (1 KB reserved each)
    static_assert(Tr::SMEM_FIXED + 64 * sizeof(real) <= kMaxSmem, "fused tile does not fit in shared memory");
    // the attribute is per device, not per process; contexts on several host threads may get here together (setting it
    // twice is harmless, the flag only saves the call)
    static std::atomic<bool> attr_set[kMaxDevices];
    if (c->device >= kMaxDevices || !attr_set[c->device].load(std::memory_order_acquire)) {
        CU_TRY(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kMaxSmem));
        if (c->device < kMaxDevices) attr_set[c->device].store(true, std::memory_order_release);
    }
    int rc = plan_fused<real, T, BX, BY, NT, PF, MINB>(c, ctas_per_sm, &P.tiles_x, &P.tiles_y, &P.bz, &P.nchunks, nullptr);
    if (rc) return rc;
    const long long units = (long long)P.tiles_x * P.tiles_y * c->g.batch;
    constexpr int H = Tr::H;
    const long long grid = units * P.nchunks;
    if (grid > 0x7fffffffLL) return fail(c, TDSE_EINVAL, "fused grid too large");
    const size_t smem = Tr::SMEM_FIXED + (size_t)(P.bz + 2 * H + 2) * sizeof(real);
    const CUtensorMap* maps = nullptr;
    rc = get_tensor_maps(c, Tr::W, Tr::NP, &maps);
    if (rc) return rc;
    const int in = c->cur;                              // maps: R[0], I[0], V, R[1], I[1]
    // Programmatic dependent launch: the next launch's CTAs may become resident and run their shared-memory
    // prologue while this one drains; the kernel orders every global access behind griddepcontrol.wait.
    cudaLaunchConfig_t lc = {};
    lc.gridDim = dim3((unsigned)grid); lc.blockDim = dim3(NT); lc.dynamicSmemBytes = smem; lc.stream = c->stream;
    cudaLaunchAttribute la[1];
    la[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    la[0].val.programmaticStreamSerializationAllowed = c->opt_pdl ? 1 : 0;
    lc.attrs = la; lc.numAttrs = 1;
    CU_TRY(c, cudaLaunchKernelEx(&lc, kern, P, maps[in ? 3 : 0], maps[in ? 4 : 1], maps[2]));
    c->launches++;
    c->last_tile_x = BX; c->last_tile_y = BY; c->last_chunks = P.nchunks;
    return TDSE_OK;
}

// The iteration barrier as a split arrive / wait mbarrier (SPLIT, tdse_kernels_fused.cuh) pays where a launch is a single wave
// of short z chunks, i.e. where skew between warps is not hidden by other CTAs' work queued behind: measured +5 % on one
// 128^3 f64 grid, +2 % on 64^3 f64, -1..2 % on every multi-wave grid and on the f32 kernels (profiles/README.md, round 2).
// tdse_set_option("variant", 1 | 2) forces it on | off.
template <typename real, int T, int BX, int BY, int NT, int PF>
bool want_split(tdse_ctx* c)
{
    if (c->opt_variant == 1) return true;
    if (c->opt_variant == 2) return false;
    if (sizeof(real) != 8) return false;
    int tx, ty, bz, nch;
    if (plan_fused<real, T, BX, BY, NT, PF>(c, 1, &tx, &ty, &bz, &nch, nullptr)) return false;
    return (long long)tx * ty * nch * c->g.batch <= c->num_sms;
}

// default prefetch depth: the launcher picks the barrier scheme (SPLIT)
template <typename real, int T, int BX, int BY, int NT, int PF, bool GHOSTXY>
int launch_fused_default(tdse_ctx* c, FusedParams& P)
{
    return want_split<real, T, BX, BY, NT, PF>(c) ? launch_fused_cfg<real, T, BX, BY, NT, PF, GHOSTXY, 1, true>(c, P, 1)
                                                  : launch_fused_cfg<real, T, BX, BY, NT, PF, GHOSTXY, 1, false>(c, P, 1);
}

template <bool GHOSTXY>
int launch_fused_bc(tdse_ctx* c, FusedParams& P, int T)
{
    if (c->dtype == TDSE_F32) {
        if (T == 2) return c->opt_pf == 1 ? launch_fused_cfg<float, 2, 64, 32, 384, 1, GHOSTXY>(c, P, 1)
                                          : launch_fused_default<float, 2, 64, 32, 384, 2, GHOSTXY>(c, P);
        return c->opt_pf == 1 ? launch_fused_cfg<float, 1, 64, 32, 352, 1, GHOSTXY>(c, P, 1)
             : c->opt_pf == 2 ? launch_fused_cfg<float, 1, 64, 32, 352, 2, GHOSTXY>(c, P, 1)
                              : launch_fused_default<float, 1, 64, 32, 352, 4, GHOSTXY>(c, P);
    }
    if (T == 2) return c->opt_pf == 1 ? launch_fused_cfg<double, 2, 32, 24, 320, 1, GHOSTXY>(c, P, 1)
                     : c->opt_pf == 2 ? launch_fused_cfg<double, 2, 32, 24, 320, 2, GHOSTXY>(c, P, 1)
                                      : launch_fused_default<double, 2, 32, 24, 320, 3, GHOSTXY>(c, P);
    return c->opt_pf == 1 ? launch_fused_cfg<double, 1, 32, 32, 352, 1, GHOSTXY>(c, P, 1)
         : c->opt_pf == 2 ? launch_fused_cfg<double, 1, 32, 32, 352, 2, GHOSTXY>(c, P, 1)
                          : launch_fused_default<double, 1, 32, 32, 352, 4, GHOSTXY>(c, P);
}

int launch_fused(tdse_ctx* c, FusedParams& P, int T)
{
    P.cxf = (float)P.cx; P.cyf = (float)P.cy; P.czf = (float)P.cz; P.cvf = (float)P.cv;
    P.c2f = (float)(2.0 * (P.cx + P.cy + P.cz));
    P.entry_bytes = (unsigned long long)c->g.pcells * c->w;
    P.px = c->g.px; P.py = c->g.py;
    const bool ghostxy = c->g.bcx == BC_DIRICHLET || c->g.bcy == BC_DIRICHLET;
    return ghostxy ? launch_fused_bc<true>(c, P, T) : launch_fused_bc<false>(c, P, T);
}

bool fused_supported(const tdse_ctx* c)
{
    const int vw = (int)(16 / c->w);
    // 16-byte vectors along x; per-entry byte offsets are 32-bit inside the fused kernel
    // (also: even ny for the row-pair view, a domain at least as wide as the frame so that images are first images)
    return c->pingpong && (c->g.nx % vw == 0) && (c->g.ny % 2 == 0) && c->g.nx >= 2 * PADX && c->g.ny >= 2 * PADY &&
           ((unsigned long long)c->g.pcells * c->w < (1ull << 32));
}

// Temporal block when the caller leaves it open.  Two steps per pass halve the traffic but march 4 more halo planes
// per chunk at 1.5x the time per plane; on grids so small that a chunk is a few planes (64^3) that costs more than
// it saves.  Estimated time per step = (a_T + b_T * planes marched per CTA) / T with the constants measured on one
// B200 (profiles/README.md, capture D: b = 0.77 / 1.16 us per plane for T = 1 / 2; a = 1.5 / 2.0 us with dependent
// launch); T = 1 is taken only when it wins by 15 %, the accuracy of this model.
int auto_tblock(tdse_ctx* c)
{
    int tx, ty, bz, nch;
    long long p1 = 0, p2 = 0;
    int rc1, rc2;
    if (c->dtype == TDSE_F32) {
        rc1 = plan_fused<float, 1, 64, 32, 352, 4>(c, 1, &tx, &ty, &bz, &nch, &p1);
        rc2 = plan_fused<float, 2, 64, 32, 384, 2>(c, 1, &tx, &ty, &bz, &nch, &p2);
    } else {
        rc1 = plan_fused<double, 1, 32, 32, 352, 4>(c, 1, &tx, &ty, &bz, &nch, &p1);
        rc2 = plan_fused<double, 2, 32, 24, 320, 3>(c, 1, &tx, &ty, &bz, &nch, &p2);
    }
    if (rc1 || rc2) return 2;
    const double t1 = 1.5 + 0.77 * (double)p1, t2 = (2.0 + 1.16 * (double)p2) / 2.0;
    return t1 < 0.85 * t2 ? 1 : 2;
}

template <typename real>
int launch_twopass_step(tdse_ctx* c)
{
    // z segments: enough blocks to fill the machine a few times over, at least 8 planes per segment
    const long long cols = (long long)((c->g.nx + 31) / 32) * ((c->g.ny + 7) / 8) * c->g.batch;
    int nseg = (int)std::min<long long>(std::max(1, c->g.nz / 8), std::max<long long>(1, (8LL * c->num_sms + cols - 1) / cols));
    nseg = (int)std::min<long long>(nseg, std::max<long long>(1, 65535 / c->g.batch));
    const int zs = (c->g.nz + nseg - 1) / nseg;
    nseg = (c->g.nz + zs - 1) / zs;
    if ((long long)c->g.batch * nseg > 65535) return fail(c, TDSE_EINVAL, "two-pass launch: batch too large for one grid");
    const dim3 grid((unsigned)((c->g.nx + 31) / 32), (unsigned)((c->g.ny + 7) / 8), (unsigned)(c->g.batch * nseg));
    const dim3 block(32, 8);
    real* R = static_cast<real*>(c->R[c->cur]);
    real* I = static_cast<real*>(c->I[c->cur]);
    const real* V = static_cast<const real*>(c->V);
    const real* M = static_cast<const real*>(c->mask_dev);
    half_step_kernel<real><<<grid, block, 0, c->stream>>>(c->g, (real)c->m.cx, (real)c->m.cy, (real)c->m.cz, (real)c->m.cv, (real)1, zs, nseg, V, M, R, I);
    CU_LAUNCH_CHECK(c);
    half_step_kernel<real><<<grid, block, 0, c->stream>>>(c->g, (real)c->m.cx, (real)c->m.cy, (real)c->m.cz, (real)c->m.cv, (real)-1, zs, nseg, V, M, I, R);
    CU_LAUNCH_CHECK(c);
    return TDSE_OK;
}

// Streamed frame mode: the ring slot the next frame goes to (NULL once the host buffer is full).  The compute stream first
// waits until the copy that last used this slot has left it.
int stream_frame_begin(tdse_ctx* c, double** frame, bool* waited)
{
    *frame = nullptr;
    *waited = false;
    if (c->nframes >= c->fs_capacity) return TDSE_OK;
    const int slot = c->nframes % c->fs_slots;
    if (c->fs_busy[slot]) { CU_TRY(c, cudaStreamWaitEvent(c->stream, c->fs_copied[slot], 0)); *waited = true; }
    *frame = c->fs_ring + (size_t)slot * c->g.batch * c->g.plane;
    return TDSE_OK;
}

// ... and its way out: once the detector kernel has written the slot, one strided copy on the second stream puts entry b's
// frame at frames_host[(b * capacity + nframes) * ny * nx] (one cudaMemcpy2DAsync per slot: rows = entries).
int stream_frame_end(tdse_ctx* c, double* frame)
{
    if (frame) {
        const int slot = c->nframes % c->fs_slots;
        const size_t plane_bytes = (size_t)c->g.plane * sizeof(double);
        CU_TRY(c, cudaEventRecord(c->fs_written[slot], c->stream));
        CU_TRY(c, cudaStreamWaitEvent(c->fs_stream, c->fs_written[slot], 0));
        if (c->fs_copy2d) {
            CU_TRY(c, cudaMemcpy2DAsync(c->fs_host + (size_t)c->nframes * c->g.plane, (size_t)c->fs_capacity * plane_bytes, frame, plane_bytes,
                                        plane_bytes, (size_t)c->g.batch, cudaMemcpyDeviceToHost, c->fs_stream));
        } else {      // host pitch capacity * plane beyond what a 2-D copy takes (cudaDevAttrMaxPitch): one copy per entry
            for (int b = 0; b < c->g.batch; ++b)
                CU_TRY(c, cudaMemcpyAsync(c->fs_host + ((size_t)b * c->fs_capacity + c->nframes) * c->g.plane, frame + (size_t)b * c->g.plane,
                                          plane_bytes, cudaMemcpyDeviceToHost, c->fs_stream));
        }
        CU_TRY(c, cudaEventRecord(c->fs_copied[slot], c->fs_stream));
        c->fs_busy[slot] = 1;
    }
    c->nframes++;
    return TDSE_OK;
}

void free_frame_stream(tdse_ctx* c)
{
    if (c->fs_stream) cudaStreamSynchronize(c->fs_stream);
    if (c->fs_ring) cudaFree(c->fs_ring);
    for (cudaEvent_t e : c->fs_written) cudaEventDestroy(e);
    for (cudaEvent_t e : c->fs_copied) cudaEventDestroy(e);
    if (c->fs_stream) cudaStreamDestroy(c->fs_stream);
    c->fs_ring = nullptr; c->fs_host = nullptr; c->fs_stream = nullptr;
    c->fs_written.clear(); c->fs_copied.clear(); c->fs_busy.clear();
    c->fs_slots = c->fs_capacity = 0;
}

// one launch per sample (accumulate + trace), programmatically serialised behind the step kernel
template <typename real>
int launch_detector(tdse_ctx* c, double* D, double* partial, double* frame, long long frame_entry_stride, int slot,
                    bool allow_pdl = true)
{
    const unsigned nblk = (unsigned)((c->g.plane + 255) / 256);
    cudaLaunchConfig_t lc = {};
    lc.gridDim = dim3(nblk, (unsigned)c->g.batch); lc.blockDim = dim3(256); lc.dynamicSmemBytes = 0; lc.stream = c->stream;
    cudaLaunchAttribute la[1];
    la[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    // griddepcontrol.wait orders this kernel behind the preceding KERNEL only.  When the stream has just been told to wait
    // for a ring slot's copy-out event, the launch must be a plain, fully stream-ordered one: nothing may touch the slot early.
    la[0].val.programmaticStreamSerializationAllowed = (c->opt_pdl && allow_pdl) ? 1 : 0;
    lc.attrs = la; lc.numAttrs = 1;
    CU_TRY(c, cudaLaunchKernelEx(&lc, detector_accum_kernel<real>, c->g, c->k_det, static_cast<const real*>(c->R[c->cur]),
                                 static_cast<const real*>(c->I[c->cur]), D, partial, frame, frame_entry_stride,
                                 c->done, c->m.dx * c->m.dy, c->trace, c->max_samples, slot));
    c->launches++;
    return TDSE_OK;
}

template <typename real>
int sample_detector(tdse_ctx* c)
{
    const unsigned nblk = (unsigned)((c->g.plane + 255) / 256);
    int rc = ensure_partial(c, (size_t)nblk * c->g.batch);
    if (rc) return rc;
    if (!c->done) {
        CU_TRY(c, cudaMalloc(&c->done, (size_t)c->g.batch * sizeof(unsigned)));
        CU_TRY(c, cudaMemsetAsync(c->done, 0, (size_t)c->g.batch * sizeof(unsigned), c->stream));
    }
    if (c->fs_ring) {
        double* frame = nullptr;
        bool waited = false;
        rc = stream_frame_begin(c, &frame, &waited);
        if (rc) return rc;
        rc = launch_detector<real>(c, c->D, c->partial, frame, c->g.plane, c->nsamples, !waited);
        if (rc) return rc;
        if ((rc = stream_frame_end(c, frame))) return rc;
    } else {
        double* frame = (c->frames && c->nframes < c->max_frames) ? c->frames + (size_t)c->nframes * c->g.plane : nullptr;
        rc = launch_detector<real>(c, c->D, c->partial, frame, (long long)c->max_frames * c->g.plane, c->nsamples);
        if (rc) return rc;
        if (c->frames) c->nframes++;
    }
    c->nsamples++;
    return TDSE_OK;
}

// frame mode: rho(0) from the state in memory before the first step
template <typename real>
int sample_initial_frame(tdse_ctx* c)
{
    if (c->fs_ring) {
        double* frame = nullptr;
        bool waited = false;
        int rc = stream_frame_begin(c, &frame, &waited);
        if (rc) return rc;
        if ((rc = launch_detector<real>(c, nullptr, nullptr, frame, c->g.plane, 0, !waited))) return rc;
        return stream_frame_end(c, frame);
    }
    const int rc = launch_detector<real>(c, nullptr, nullptr, c->frames, (long long)c->max_frames * c->g.plane, 0);
    if (rc) return rc;
    c->nframes = 1;
    return TDSE_OK;
}

}  // namespace

// =================================================================================================
// C ABI
// =================================================================================================
extern "C" {

const char* tdse_last_error(const tdse_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

size_t tdse_workspace_bytes(int nx, int ny, int nz, int batch, int dtype, int pingpong)
{
    if (nx < 1 || ny < 1 || nz < 1 || batch < 1 || (dtype != TDSE_F32 && dtype != TDSE_F64)) return 0;
    const size_t arr = align_up((size_t)(nx + 2 * PADX) * (ny + 2 * PADY) * nz * batch * elem_bytes(dtype));
    return (pingpong ? 5 : 3) * arr;
}

int tdse_create(tdse_ctx** out, int nx, int ny, int nz, int batch,
                double dx, double dt, double mass, double hbar, int dtype)
{
    if (!out) return fail(nullptr, TDSE_EINVAL, "tdse_create: out is NULL");
    if (nx < 1 || ny < 1 || nz < 1 || batch < 1) return fail(nullptr, TDSE_EINVAL, "tdse_create: sizes must be >= 1");
    if (!(dx > 0) || !(dt > 0) || !(mass > 0) || !(hbar > 0)) return fail(nullptr, TDSE_EINVAL, "tdse_create: dx, dt, mass, hbar must be > 0");
    if (dtype != TDSE_F32 && dtype != TDSE_F64) return fail(nullptr, TDSE_EINVAL, "tdse_create: unknown dtype");
    if ((long long)nx * ny > 0x3fffffffLL) return fail(nullptr, TDSE_EINVAL, "tdse_create: nx*ny too large");
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(nullptr, TDSE_ECUDA, std::string("tdse_create: no CUDA device (") + cudaGetErrorString(e) + "); libtdse has no CPU fallback");
    }
    tdse_ctx* c = new (std::nothrow) tdse_ctx();
    if (!c) return fail(nullptr, TDSE_ENOMEM, "tdse_create: out of host memory");
    c->g.nx = nx; c->g.ny = ny; c->g.nz = nz; c->g.batch = batch;
    c->g.bcx = c->g.bcy = c->g.bcz = BC_PERIODIC;
    c->g.plane = (long long)nx * ny;
    c->g.cells = c->g.plane * nz;
    c->g.px = nx + 2 * PADX; c->g.py = ny + 2 * PADY;
    c->g.pplane = (long long)c->g.px * c->g.py;
    c->g.pcells = c->g.pplane * nz;
    c->dtype = dtype; c->w = elem_bytes(dtype);
    c->dx = dx; c->dt = dt; c->mass = mass; c->hbar = hbar;
    c->m.dx = c->m.dy = c->m.dz = dx;
    c->m.cx = c->m.cy = c->m.cz = hbar * dt / (2.0 * mass * dx * dx);
    c->m.cv = dt / hbar;
    c->arr_bytes = align_up((size_t)c->g.pcells * batch * c->w);
    c->have_V.assign(batch, 0);
    c->have_state.assign(batch, 0);
    auto bail = [&](const char* what, cudaError_t err) {
        std::string m = std::string("tdse_create: ") + what + ": " + cudaGetErrorString(err);
        tdse_destroy(c);
        return fail(nullptr, TDSE_ECUDA, m);
    };
    if ((e = cudaGetDevice(&c->device)) != cudaSuccess) return bail("cudaGetDevice", e);
    if ((e = cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, c->device)) != cudaSuccess) return bail("SM count", e);
    if ((e = cudaMalloc(&c->D, (size_t)batch * c->g.plane * sizeof(double))) != cudaSuccess) return bail("detector image", e);
    if ((e = cudaMalloc(&c->scalars, 4 * sizeof(double))) != cudaSuccess) return bail("scalars", e);
    if ((e = cudaEventCreateWithFlags(&c->atoms_ev, cudaEventDisableTiming)) != cudaSuccess) return bail("event", e);
    int rc = upload_mask(c);
    if (rc) { std::string m = c->err; tdse_destroy(c); return fail(nullptr, rc, m); }
    rc = reset_detector(c);
    if (rc) { std::string m = c->err; tdse_destroy(c); return fail(nullptr, rc, m); }
    *out = c;
    return TDSE_OK;
}

int tdse_destroy(tdse_ctx* c)
{
    if (!c) return TDSE_OK;
    DeviceScope on_device_(c);      // frees what it can even if the switch failed
    cudaStreamSynchronize(c->stream);
    if (c->ws_owned && c->ws) cudaFree(c->ws);
    if (c->mask_dev) cudaFree(c->mask_dev);
    if (c->D) cudaFree(c->D);
    if (c->trace) cudaFree(c->trace);
    if (c->frames) cudaFree(c->frames);
    free_frame_stream(c);
    if (c->partial) cudaFree(c->partial);
    if (c->done) cudaFree(c->done);
    if (c->scalars) cudaFree(c->scalars);
    if (c->cell_stage) cudaFree(c->cell_stage);
    if (c->pot_ranges) cudaFree(c->pot_ranges);
    if (c->pot_count) cudaFree(c->pot_count);
    if (c->pot_prefix) cudaFree(c->pot_prefix);
    if (c->atoms_dev) cudaFree(c->atoms_dev);
    if (c->atoms_pin) cudaFreeHost(c->atoms_pin);
    if (c->atoms_ev) cudaEventDestroy(c->atoms_ev);
    cudaGetLastError();
    delete c;
    return TDSE_OK;
}

int tdse_bind(tdse_ctx* c, void* dev_workspace, size_t bytes, void* cuda_stream)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    if (!dev_workspace) return fail(c, TDSE_EINVAL, "tdse_bind: workspace is NULL");
    if (reinterpret_cast<uintptr_t>(dev_workspace) % kAlign) return fail(c, TDSE_EINVAL, "tdse_bind: workspace must be 256-byte aligned");
    if (bytes < 3 * c->arr_bytes) return fail(c, TDSE_ENOMEM, "tdse_bind: workspace smaller than tdse_workspace_bytes(..., 0)");
    cudaStreamSynchronize(c->stream);
    if (c->ws_owned && c->ws) cudaFree(c->ws);
    c->ws = dev_workspace; c->ws_bytes = bytes; c->ws_owned = false;
    c->pingpong = bytes >= 5 * c->arr_bytes;
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    carve(c);
    CU_TRY(c, cudaMemsetAsync(c->ws, 0, (c->pingpong ? 5 : 3) * c->arr_bytes, c->stream));   // frames of Dirichlet axes stay zero
    return reset_detector(c);
}

int tdse_set_boundary(tdse_ctx* c, int bcx, int bcy, int bcz, int absorb_lo, int absorb_hi, double strength, int power)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    auto okbc = [](int b) { return b == TDSE_BC_PERIODIC || b == TDSE_BC_DIRICHLET; };
    if (!okbc(bcx) || !okbc(bcy) || !okbc(bcz)) return fail(c, TDSE_EINVAL, "tdse_set_boundary: unknown boundary flag");
    if (absorb_lo < 0 || absorb_hi < 0 || absorb_lo + absorb_hi > c->g.nz) return fail(c, TDSE_EINVAL, "tdse_set_boundary: absorber widths");
    if (!(strength >= 0.0 && strength <= 1.0) || power < 1) return fail(c, TDSE_EINVAL, "tdse_set_boundary: strength in [0,1], power >= 1");
    const bool xy_changed = bcx != c->g.bcx || bcy != c->g.bcy;
    c->g.bcx = bcx; c->g.bcy = bcy; c->g.bcz = bcz;
    c->absorb_lo = absorb_lo; c->absorb_hi = absorb_hi; c->strength = strength; c->power = power;
    int rc = upload_mask(c);
    if (rc) return rc;
    // The storage frame of every xy plane holds periodic images or Dirichlet zeros (tdse_common.cuh) and the fused kernel
    // takes its x/y neighbours from it: data loaded under the old flags gets the frame of the new ones.
    if (xy_changed && c->ws) {
        for (int e = 0; e < c->g.batch; ++e) {
            if (c->have_V[e] && (rc = fill_frame(c, entry_ptr(c, c->V, e)))) return rc;
            if (c->have_state[e]) {
                if ((rc = fill_frame(c, entry_ptr(c, c->R[c->cur], e)))) return rc;
                if ((rc = fill_frame(c, entry_ptr(c, c->I[c->cur], e)))) return rc;
            }
        }
    }
    return TDSE_OK;
}

}  // extern "C"

namespace {

// host atom list -> pinned staging buffer -> device copy (both library-owned, grown on demand), asynchronously
int stage_atoms(tdse_ctx* c, const AtomRec* atoms_host, int natoms)
{
    static_assert(sizeof(AtomRec) == sizeof(tdse_atom), "atom record layout");
    if (natoms > c->atoms_cap) {
        CU_TRY(c, cudaStreamSynchronize(c->stream));
        if (c->atoms_dev) cudaFree(c->atoms_dev);
        if (c->atoms_pin) cudaFreeHost(c->atoms_pin);
        c->atoms_dev = nullptr; c->atoms_pin = nullptr; c->atoms_cap = 0;
        const int cap = std::max(natoms, 1024);
        CU_TRY(c, cudaMalloc(&c->atoms_dev, (size_t)cap * sizeof(AtomRec)));
        CU_TRY(c, cudaMallocHost(&c->atoms_pin, (size_t)cap * sizeof(AtomRec)));
        c->atoms_cap = cap;
        c->atoms_pending = false;
    }
    if (c->atoms_pending) { CU_TRY(c, cudaEventSynchronize(c->atoms_ev)); c->atoms_pending = false; }
    if (natoms > 0) {
        std::memcpy(c->atoms_pin, atoms_host, (size_t)natoms * sizeof(AtomRec));
        CU_TRY(c, cudaMemcpyAsync(c->atoms_dev, c->atoms_pin, (size_t)natoms * sizeof(AtomRec), cudaMemcpyHostToDevice, c->stream));
        // the pinned staging buffer may be rewritten once this copy is done (event); the device copy is
        // rewritten by the next call's H2D, which the stream orders after this call's build kernel
        CU_TRY(c, cudaEventRecord(c->atoms_ev, c->stream));
        c->atoms_pending = true;
    }
    return TDSE_OK;
}

// One launch of the potential builder: entries e0 .. e0+nent-1, entry q sums atoms [first, first+count) of `atoms_dev`
// (ranges_dev[q], or (first0, count0) for every entry when ranges_dev is NULL), starting from prefix_in if given.
template <typename real, int CELLS, bool HAS_CUT, bool PREFIX_OUT>
int launch_potential(tdse_ctx* c, int e0, int nent, const AtomRec* atoms_dev, const AtomRange* ranges_dev, int first0,
                            int count0, const double* prefix_in, double vmin, double vmax, double rcut, double* prefix_out)
{
    const long long bricks = (long long)((c->g.nx + CELLS * kPotBX - 1) / (CELLS * kPotBX)) *
                             ((c->g.ny + kPotBY - 1) / kPotBY) * ((c->g.nz + kPotBZ - 1) / kPotBZ);
    if (bricks > 0x7fffffffLL || nent > 65535) return fail(c, TDSE_EINVAL, "tdse_set_potential: grid too large");
    potential_build_kernel<real, CELLS, HAS_CUT, PREFIX_OUT><<<dim3((unsigned)bricks, (unsigned)nent), 256, 0, c->stream>>>(
        c->g, c->m.dx, c->m.dy, c->m.dz, atoms_dev, ranges_dev, first0, count0, prefix_in, vmin, vmax, rcut,
        reinterpret_cast<real*>(entry_ptr(c, c->V, e0)), prefix_out);
    CU_LAUNCH_CHECK(c);
    return TDSE_OK;
}

template <bool PREFIX_OUT>
int launch_potential_any(tdse_ctx* c, int e0, int nent, const AtomRec* atoms_dev, const AtomRange* ranges_dev, int first0,
                                int count0, const double* prefix_in, double vmin, double vmax, double rcut, double* prefix_out)
{
    const bool wide = c->g.nx >= 8 * kPotBX;       // 8 cells per thread once a brick row of 128 cells fits
    const bool cut = rcut > 0.0;
#define TDSE_POT(REAL, CELLS, CUT) \
    launch_potential<REAL, CELLS, CUT, PREFIX_OUT>(c, e0, nent, atoms_dev, ranges_dev, first0, count0, prefix_in, vmin, vmax, rcut, prefix_out)
    if (c->dtype == TDSE_F32) {
        if (wide) return cut ? TDSE_POT(float, 8, true) : TDSE_POT(float, 8, false);
        return cut ? TDSE_POT(float, 4, true) : TDSE_POT(float, 4, false);
    }
    if (wide) return cut ? TDSE_POT(double, 8, true) : TDSE_POT(double, 8, false);
    return cut ? TDSE_POT(double, 4, true) : TDSE_POT(double, 4, false);
#undef TDSE_POT
}

// one atom list for entries b0 .. b1-1 (built once, copied to the others)
int build_potential(tdse_ctx* c, int b, const AtomRec* atoms_dev, int natoms, double vmin, double vmax, double rcut)
{
    int b0, b1;
    if (!entry_range(c, b, &b0, &b1)) return fail(c, TDSE_EINVAL, "tdse_set_potential: entry out of range");
    const int rc = launch_potential_any<false>(c, b0, 1, atoms_dev, nullptr, 0, natoms, nullptr, vmin, vmax, rcut, nullptr);
    if (rc) return rc;
    void* dst = entry_ptr(c, c->V, b0);
    for (int e = b0 + 1; e < b1; ++e)
        CU_TRY(c, cudaMemcpyAsync(entry_ptr(c, c->V, e), dst, (size_t)c->g.pcells * c->w, cudaMemcpyDeviceToDevice, c->stream));
    for (int e = b0; e < b1; ++e) c->have_V[e] = 1;
    c->vabs_max = std::max(c->vabs_max, std::max(std::fabs(vmin), std::fabs(vmax)));
    return TDSE_OK;
}

// every entry its own list, one launch; the atoms all lists start with (nshared) are summed once into an fp64 scratch
int build_potential_batch(tdse_ctx* c, const AtomRec* atoms_dev, const std::vector<AtomRange>& ranges, int nshared,
                                 double vmin, double vmax, double rcut)
{
    const int batch = c->g.batch;
    if (!c->pot_ranges) CU_TRY(c, cudaMalloc(&c->pot_ranges, (size_t)batch * sizeof(AtomRange)));
    std::vector<AtomRange> rest(ranges);
    const double* prefix = nullptr;
    // sharing pays when the prefix pass (one entry's worth of work on nshared atoms) is cheaper than what it saves
    if (batch >= 2 && nshared >= 8) {
        if (!c->pot_prefix) {
            const cudaError_t e = cudaMalloc(&c->pot_prefix, (size_t)c->g.cells * sizeof(double));
            if (e != cudaSuccess) { cudaGetLastError(); c->pot_prefix = nullptr; }     // no scratch: plain sums
        }
        if (c->pot_prefix) {
            const int rc = launch_potential_any<true>(c, 0, 1, atoms_dev, nullptr, ranges[0].first, nshared, nullptr, vmin, vmax, rcut, c->pot_prefix);
            if (rc) return rc;
            for (AtomRange& r : rest) { r.first += nshared; r.count -= nshared; }
            prefix = c->pot_prefix;
        }
    }
    // the previous call's ranges may still be in use by its kernel: the copy is ordered behind it on the stream
    // (pageable source: cudaMemcpyAsync returns once `rest` has been staged)
    CU_TRY(c, cudaMemcpyAsync(c->pot_ranges, rest.data(), (size_t)batch * sizeof(AtomRange), cudaMemcpyHostToDevice, c->stream));
    const int rc = launch_potential_any<false>(c, 0, batch, atoms_dev, c->pot_ranges, 0, 0, prefix, vmin, vmax, rcut, nullptr);
    if (rc) return rc;
    std::fill(c->have_V.begin(), c->have_V.end(), 1);
    c->vabs_max = std::max(c->vabs_max, std::max(std::fabs(vmin), std::fabs(vmax)));
    return TDSE_OK;
}

}  // namespace

extern "C" {

int tdse_set_spacing(tdse_ctx* c, double dy, double dz)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    if (!(dy > 0) || !(dz > 0)) return fail(c, TDSE_EINVAL, "tdse_set_spacing: dy, dz must be > 0");
    c->m.dy = dy; c->m.dz = dz;
    c->m.cy = c->hbar * c->dt / (2.0 * c->mass * dy * dy);
    c->m.cz = c->hbar * c->dt / (2.0 * c->mass * dz * dz);
    // potential and state were built on the old mesh
    std::fill(c->have_V.begin(), c->have_V.end(), 0);
    std::fill(c->have_state.begin(), c->have_state.end(), 0);
    c->vabs_max = 0.0;
    return reset_detector(c);
}

int tdse_set_potential(tdse_ctx* c, int b, const tdse_atom* atoms_host, int natoms, double vmin, double vmax, double rcut)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    if (natoms < 0 || (natoms > 0 && !atoms_host)) return fail(c, TDSE_EINVAL, "tdse_set_potential: atom list");
    if (!(vmin <= vmax)) return fail(c, TDSE_EINVAL, "tdse_set_potential: vmin > vmax");
    int rc = ensure_workspace(c);
    if (rc) return rc;
    rc = stage_atoms(c, reinterpret_cast<const AtomRec*>(atoms_host), natoms);
    if (rc) return rc;
    return build_potential(c, b, c->atoms_dev, natoms, vmin, vmax, rcut);
}

int tdse_set_potential_device(tdse_ctx* c, int b, const tdse_atom* atoms_device, int natoms, double vmin, double vmax, double rcut)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    if (natoms < 0 || (natoms > 0 && !atoms_device)) return fail(c, TDSE_EINVAL, "tdse_set_potential_device: atom list");
    if (!(vmin <= vmax)) return fail(c, TDSE_EINVAL, "tdse_set_potential_device: vmin > vmax");
    int rc = ensure_workspace(c);
    if (rc) return rc;
    return build_potential(c, b, reinterpret_cast<const AtomRec*>(atoms_device), natoms, vmin, vmax, rcut);
}

int tdse_set_potential_batch(tdse_ctx* c, const tdse_atom* atoms, const int* offsets_host, int on_device,
                             double vmin, double vmax, double rcut)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    const int batch = c->g.batch;
    if (!offsets_host) return fail(c, TDSE_EINVAL, "tdse_set_potential_batch: offsets is NULL");
    if (!(vmin <= vmax)) return fail(c, TDSE_EINVAL, "tdse_set_potential_batch: vmin > vmax");
    std::vector<AtomRange> ranges(batch);
    for (int e = 0; e < batch; ++e) {
        if (offsets_host[e] < 0 || offsets_host[e + 1] < offsets_host[e])
            return fail(c, TDSE_EINVAL, "tdse_set_potential_batch: offsets must be non-negative and non-decreasing");
        ranges[e].first = offsets_host[e];
        ranges[e].count = offsets_host[e + 1] - offsets_host[e];
    }
    const int total = offsets_host[batch];
    if (total > 0 && !atoms) return fail(c, TDSE_EINVAL, "tdse_set_potential_batch: atom list");
    int rc = ensure_workspace(c);
    if (rc) return rc;
    int min_count = ranges[0].count;
    for (const AtomRange& r : ranges) min_count = std::min(min_count, r.count);
    int nshared = 0;
    const AtomRec* atoms_dev = reinterpret_cast<const AtomRec*>(atoms);
    if (!on_device) {
        const AtomRec* host = reinterpret_cast<const AtomRec*>(atoms);
        nshared = batch >= 2 ? min_count : 0;
        for (int e = 1; e < batch && nshared > 0; ++e)
            for (int a = 0; a < nshared; ++a)
                if (std::memcmp(host + ranges[0].first + a, host + ranges[e].first + a, sizeof(AtomRec)) != 0) { nshared = a; break; }
        rc = stage_atoms(c, host, total);
        if (rc) return rc;
        atoms_dev = c->atoms_dev;
    } else if (batch >= 2 && min_count >= 8) {
        // shared prefix of device-resident lists: compared on the device, one int comes back
        if (!c->pot_ranges) CU_TRY(c, cudaMalloc(&c->pot_ranges, (size_t)batch * sizeof(AtomRange)));
        if (!c->pot_count) CU_TRY(c, cudaMalloc(&c->pot_count, sizeof(int)));
        CU_TRY(c, cudaMemcpyAsync(c->pot_ranges, ranges.data(), (size_t)batch * sizeof(AtomRange), cudaMemcpyHostToDevice, c->stream));
        CU_TRY(c, cudaMemcpyAsync(c->pot_count, &min_count, sizeof(int), cudaMemcpyHostToDevice, c->stream));
        common_prefix_kernel<<<dim3((unsigned)((min_count + 127) / 128), (unsigned)(batch - 1)), 128, 0, c->stream>>>(
            atoms_dev, c->pot_ranges, min_count, c->pot_count);
        CU_LAUNCH_CHECK(c);
        CU_TRY(c, cudaMemcpyAsync(&nshared, c->pot_count, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
        CU_TRY(c, cudaStreamSynchronize(c->stream));
    }
    return build_potential_batch(c, atoms_dev, ranges, nshared, vmin, vmax, rcut);
}

int tdse_set_potential_cell(tdse_ctx* c, int b, const double* cell, int on_device, int mx, int my, int mz,
                            double ax, double ay, double az, double x0, double y0, double z0, double vmin, double vmax)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    if (!cell || mx < 1 || my < 1 || mz < 1) return fail(c, TDSE_EINVAL, "tdse_set_potential_cell: cell grid");
    if (!(ax > 0) || !(ay > 0) || !(az > 0)) return fail(c, TDSE_EINVAL, "tdse_set_potential_cell: cell edge lengths must be > 0");
    if (!(vmin <= vmax)) return fail(c, TDSE_EINVAL, "tdse_set_potential_cell: vmin > vmax");
    int b0, b1;
    if (!entry_range(c, b, &b0, &b1)) return fail(c, TDSE_EINVAL, "tdse_set_potential_cell: entry out of range");
    int rc = ensure_workspace(c);
    if (rc) return rc;
    const size_t n = (size_t)mx * my * mz;
    const double* cell_dev = cell;
    if (!on_device) {
        // library-owned staging buffer, kept across calls (grown when a larger cell arrives); the copy and the kernel
        // are ordered on the stream, and cudaMemcpyAsync from pageable memory returns once the source has been read
        if (n > c->cell_cap) {
            if (c->cell_stage) { CU_TRY(c, cudaStreamSynchronize(c->stream)); cudaFree(c->cell_stage); c->cell_stage = nullptr; c->cell_cap = 0; }
            const cudaError_t e = cudaMalloc(&c->cell_stage, n * sizeof(double));
            if (e != cudaSuccess) { cudaGetLastError(); c->cell_stage = nullptr; return fail(c, TDSE_ENOMEM, std::string("tdse_set_potential_cell: staging: ") + cudaGetErrorString(e)); }
            c->cell_cap = n;
        }
        CU_TRY(c, cudaMemcpyAsync(c->cell_stage, cell, n * sizeof(double), cudaMemcpyHostToDevice, c->stream));
        cell_dev = c->cell_stage;
    }
    CellParams p{mx, my, mz, ax, ay, az, x0, y0, z0, vmin, vmax};
    const dim3 cgrid((unsigned)((c->g.nx + 31) / 32), (unsigned)((c->g.ny + 7) / 8), (unsigned)((c->g.nz + kCellSeg - 1) / kCellSeg));
    if (cgrid.y > 65535 || cgrid.z > 65535) return fail(c, TDSE_EINVAL, "tdse_set_potential_cell: grid too large");
    void* dst = entry_ptr(c, c->V, b0);
    if (c->dtype == TDSE_F32)
        potential_cell_kernel<float><<<cgrid, dim3(32, 8), 0, c->stream>>>(c->g, c->m.dx, c->m.dy, c->m.dz, cell_dev, p, static_cast<float*>(dst));
    else
        potential_cell_kernel<double><<<cgrid, dim3(32, 8), 0, c->stream>>>(c->g, c->m.dx, c->m.dy, c->m.dz, cell_dev, p, static_cast<double*>(dst));
    CU_LAUNCH_CHECK(c);
    for (int e = b0 + 1; e < b1; ++e)
        CU_TRY(c, cudaMemcpyAsync(entry_ptr(c, c->V, e), dst, (size_t)c->g.pcells * c->w, cudaMemcpyDeviceToDevice, c->stream));
    for (int e = b0; e < b1; ++e) c->have_V[e] = 1;
    c->vabs_max = std::max(c->vabs_max, std::max(std::fabs(vmin), std::fabs(vmax)));
    return TDSE_OK;
}

int tdse_set_potential_grid(tdse_ctx* c, int b, const void* V, int on_device)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    if (!V) return fail(c, TDSE_EINVAL, "tdse_set_potential_grid: V is NULL");
    int b0, b1;
    if (!entry_range(c, b, &b0, &b1)) return fail(c, TDSE_EINVAL, "tdse_set_potential_grid: entry out of range");
    int rc = ensure_workspace(c);
    if (rc) return rc;
    for (int e = b0; e < b1; ++e) {
        rc = copy_entry(c, entry_ptr(c, c->V, e), const_cast<void*>(V), on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, true);
        if (rc) return rc;
        rc = fill_frame(c, entry_ptr(c, c->V, e));
        if (rc) return rc;
        c->have_V[e] = 1;
    }
    // max |V| for the stability bound
    rc = ensure_partial(c, 1024);
    if (rc) return rc;
    if (c->dtype == TDSE_F32)
        absmax_partial_kernel<float><<<256, 256, 0, c->stream>>>(static_cast<const float*>((void*)entry_ptr(c, c->V, b0)), c->g.pcells, c->partial);
    else
        absmax_partial_kernel<double><<<256, 256, 0, c->stream>>>(static_cast<const double*>((void*)entry_ptr(c, c->V, b0)), c->g.pcells, c->partial);
    CU_LAUNCH_CHECK(c);
    double part[256];
    CU_TRY(c, cudaMemcpyAsync(part, c->partial, sizeof(part), cudaMemcpyDeviceToHost, c->stream));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    for (double v : part) c->vabs_max = std::max(c->vabs_max, v);
    return TDSE_OK;
}

int tdse_set_wavepacket(tdse_ctx* c, int b, double x0, double y0, double z0, double sigma,
                        double kx, double ky, double kz, double amplitude)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    if (!(sigma > 0)) return fail(c, TDSE_EINVAL, "tdse_set_wavepacket: sigma must be > 0");
    int b0, b1;
    if (!entry_range(c, b, &b0, &b1)) return fail(c, TDSE_EINVAL, "tdse_set_wavepacket: entry out of range");
    if (!c->ws) return fail(c, TDSE_ESTATE, "tdse_set_wavepacket: set the potential first (the staggered start needs V)");
    for (int e = b0; e < b1; ++e)
        if (!c->have_V[e]) return fail(c, TDSE_ESTATE, "tdse_set_wavepacket: set the potential first (the staggered start needs V)");
    const double pi = 3.14159265358979323846;
    PacketParams p;
    p.x0 = x0; p.y0 = y0; p.z0 = z0; p.inv2s2 = 1.0 / (2.0 * sigma * sigma);
    p.kx = kx; p.ky = ky; p.kz = kz;
    p.amp = amplitude != 0.0 ? amplitude : std::pow(pi * sigma * sigma, -0.75);
    const unsigned nblk = (unsigned)((c->g.cells + 255) / 256);
    // one launch for all the entries that get this packet: a thread evaluates it once and walks the entries
    if (c->dtype == TDSE_F32)
        wavepacket_init_kernel<float><<<nblk, 256, 0, c->stream>>>(c->g, c->m, p, b1 - b0,
            (const float*)entry_ptr(c, c->V, b0), (float*)entry_ptr(c, c->R[c->cur], b0), (float*)entry_ptr(c, c->I[c->cur], b0));
    else
        wavepacket_init_kernel<double><<<nblk, 256, 0, c->stream>>>(c->g, c->m, p, b1 - b0,
            (const double*)entry_ptr(c, c->V, b0), (double*)entry_ptr(c, c->R[c->cur], b0), (double*)entry_ptr(c, c->I[c->cur], b0));
    CU_LAUNCH_CHECK(c);
    for (int e = b0; e < b1; ++e) c->have_state[e] = 1;
    return reset_detector(c);
}

int tdse_set_state(tdse_ctx* c, int b, const void* R, const void* I_half, int on_device)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    if (!R || !I_half) return fail(c, TDSE_EINVAL, "tdse_set_state: NULL state");
    int b0, b1;
    if (!entry_range(c, b, &b0, &b1)) return fail(c, TDSE_EINVAL, "tdse_set_state: entry out of range");
    int rc = ensure_workspace(c);
    if (rc) return rc;
    const cudaMemcpyKind kind = on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    for (int e = b0; e < b1; ++e) {
        if ((rc = copy_entry(c, entry_ptr(c, c->R[c->cur], e), const_cast<void*>(R), kind, true))) return rc;
        if ((rc = copy_entry(c, entry_ptr(c, c->I[c->cur], e), const_cast<void*>(I_half), kind, true))) return rc;
        if ((rc = fill_frame(c, entry_ptr(c, c->R[c->cur], e)))) return rc;
        if ((rc = fill_frame(c, entry_ptr(c, c->I[c->cur], e)))) return rc;
        c->have_state[e] = 1;
    }
    if (!on_device) CU_TRY(c, cudaStreamSynchronize(c->stream));   // caller may reuse pageable buffers
    return reset_detector(c);
}

int tdse_set_detector(tdse_ctx* c, int k_plane, int every, int max_samples)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    if (every < 0 || max_samples < 0) return fail(c, TDSE_EINVAL, "tdse_set_detector: every, max_samples must be >= 0");
    if (every > 0 && (k_plane < 0 || k_plane >= c->g.nz)) return fail(c, TDSE_EINVAL, "tdse_set_detector: plane out of range");
    if (max_samples != c->max_samples) {
        // a new trace buffer is allocated before the old one is given up, so a failed allocation leaves the context usable
        double* fresh = nullptr;
        if (max_samples > 0) {
            const cudaError_t e = cudaMalloc(&fresh, (size_t)c->g.batch * max_samples * sizeof(double));
            if (e != cudaSuccess) {
                cudaGetLastError();
                return fail(c, TDSE_ENOMEM, std::string("tdse_set_detector: trace buffer: ") + cudaGetErrorString(e));
            }
        }
        if (c->trace) { CU_TRY(c, cudaStreamSynchronize(c->stream)); cudaFree(c->trace); }
        c->trace = fresh;
        c->max_samples = max_samples;
    }
    c->k_det = k_plane; c->every = every;
    return reset_detector(c);
}

int tdse_step(tdse_ctx* c, int n)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    if (n < 0) return fail(c, TDSE_EINVAL, "tdse_step: n < 0");
    if (!c->ws) return fail(c, TDSE_ESTATE, "tdse_step: potential and state are not set");
    for (int e = 0; e < c->g.batch; ++e)
        if (!c->have_V[e] || !c->have_state[e]) return fail(c, TDSE_ESTATE, "tdse_step: potential and state must be set for every entry");
    if (!c->allow_unstable) {
        // largest eigenvalue of the discrete kinetic operator: (2 hbar^2 / m) (1/dx^2 + 1/dy^2 + 1/dz^2)
        const double kin = 2.0 * c->hbar * c->hbar / c->mass *
                           (1.0 / (c->m.dx * c->m.dx) + 1.0 / (c->m.dy * c->m.dy) + 1.0 / (c->m.dz * c->m.dz));
        const double bound = 2.0 * c->hbar / (kin + c->vabs_max);
        if (c->dt > bound) {
            char buf[200];
            std::snprintf(buf, sizeof buf, "tdse_step: dt = %.6g exceeds the stability bound %.6g (max|V| = %.6g)", c->dt, bound, c->vabs_max);
            return fail(c, TDSE_EUNSTABLE, buf);
        }
    }
    int kernel = c->opt_kernel;
    if (kernel == TDSE_KERNEL_AUTO) kernel = fused_supported(c) ? TDSE_KERNEL_FUSED : TDSE_KERNEL_TWOPASS;
    if (kernel == TDSE_KERNEL_FUSED && !fused_supported(c))
        return fail(c, TDSE_EINVAL, "tdse_step: fused kernel needs a 5-array workspace, rows of whole 16-byte groups, even ny, nx >= 8 and ny >= 8");
    const int tmax = (c->opt_tblock > 0) ? c->opt_tblock : (kernel == TDSE_KERNEL_FUSED ? auto_tblock(c) : 1);
    c->last_kernel = kernel;
    if (n > 0 && (c->frames || c->fs_ring) && c->frames_t0 && c->every > 0 && c->steps == 0 && c->nframes == 0) {
        const int rc0 = (c->dtype == TDSE_F32) ? sample_initial_frame<float>(c) : sample_initial_frame<double>(c);
        if (rc0) return rc0;
    }
    int remaining = n;
    while (remaining > 0) {
        const int to_sample = (c->every > 0) ? (int)(c->every - (c->steps % c->every)) : std::numeric_limits<int>::max();
        int rc;
        if (kernel == TDSE_KERNEL_TWOPASS) {
            rc = (c->dtype == TDSE_F32) ? launch_twopass_step<float>(c) : launch_twopass_step<double>(c);
            if (rc) return rc;
            c->steps += 1; remaining -= 1;
            c->last_tblock = 1;
            if (to_sample == 1) {
                rc = (c->dtype == TDSE_F32) ? sample_detector<float>(c) : sample_detector<double>(c);
                if (rc) return rc;
            }
        } else {
            const int T = std::min(std::min(tmax, remaining), to_sample);
            const bool sample = (T == to_sample);
            FusedParams P{};
            P.Rin = c->R[c->cur]; P.Iin = c->I[c->cur]; P.V = c->V;
            P.Rout = c->R[c->cur ^ 1]; P.Iout = c->I[c->cur ^ 1];
            P.mask = c->mask_dev;
            P.nx = c->g.nx; P.ny = c->g.ny; P.nz = c->g.nz; P.batch = c->g.batch;
            P.bcx = c->g.bcx; P.bcy = c->g.bcy; P.bcz = c->g.bcz;
            P.cx = c->m.cx; P.cy = c->m.cy; P.cz = c->m.cz; P.cv = c->m.cv;
            rc = launch_fused(c, P, T);
            if (rc) return rc;
            c->cur ^= 1;
            c->steps += T; remaining -= T;
            c->last_tblock = T;
            if (sample) {   // R^s and I^{s-1/2} are exactly what the pass just wrote
                rc = (c->dtype == TDSE_F32) ? sample_detector<float>(c) : sample_detector<double>(c);
                if (rc) return rc;
            }
        }
    }
    return TDSE_OK;
}

int tdse_detector_read(tdse_ctx* c, int b, double* image_host, double* trace_host, int cap, int* nsamples)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    if (b < 0 || b >= c->g.batch) return fail(c, TDSE_EINVAL, "tdse_detector_read: entry out of range");
    if (cap < 0) return fail(c, TDSE_EINVAL, "tdse_detector_read: cap < 0");
    if (image_host)
        CU_TRY(c, cudaMemcpyAsync(image_host, c->D + (size_t)b * c->g.plane, (size_t)c->g.plane * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    const int ntr = std::min(std::min(cap, c->nsamples), c->max_samples);
    if (trace_host && ntr > 0)
        CU_TRY(c, cudaMemcpyAsync(trace_host, c->trace + (size_t)b * c->max_samples, (size_t)ntr * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    if (nsamples) *nsamples = c->nsamples;
    return TDSE_OK;
}

int tdse_set_frames(tdse_ctx* c, int max_frames, int include_t0)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    if (max_frames < 0) return fail(c, TDSE_EINVAL, "tdse_set_frames: max_frames < 0");
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    free_frame_stream(c);                // flat and streamed frame mode exclude each other
    if (c->frames) { cudaFree(c->frames); c->frames = nullptr; }
    c->max_frames = 0; c->frames_t0 = include_t0 ? 1 : 0;
    if (max_frames > 0) {
        cudaError_t e = cudaMalloc(&c->frames, (size_t)c->g.batch * max_frames * c->g.plane * sizeof(double));
        if (e != cudaSuccess) { cudaGetLastError(); c->frames = nullptr; return fail(c, TDSE_ENOMEM, std::string("tdse_set_frames: ") + cudaGetErrorString(e)); }
        c->max_frames = max_frames;
    }
    return reset_detector(c);
}

int tdse_frames_read(tdse_ctx* c, int b, int first, int count, double* frames_host, int* nframes)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    if (b < 0 || b >= c->g.batch) return fail(c, TDSE_EINVAL, "tdse_frames_read: entry out of range");
    const int have = std::min(c->nframes, c->max_frames);
    if (first < 0 || count < 0 || first + count > have) return fail(c, TDSE_EINVAL, "tdse_frames_read: frame range exceeds the frames kept");
    if (count > 0) {
        if (!frames_host) return fail(c, TDSE_EINVAL, "tdse_frames_read: NULL");
        CU_TRY(c, cudaMemcpyAsync(frames_host, c->frames + ((size_t)b * c->max_frames + first) * c->g.plane,
                                  (size_t)count * c->g.plane * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    }
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    if (nframes) *nframes = c->nframes;
    return TDSE_OK;
}

int tdse_frames_device(tdse_ctx* c, double** frames_device, int* max_frames, int* nframes)
{
    if (!c) return TDSE_EINVAL;
    if (frames_device) *frames_device = c->frames;
    if (max_frames) *max_frames = c->max_frames;
    if (nframes) *nframes = c->nframes;
    return TDSE_OK;
}

int tdse_set_frame_stream(tdse_ctx* c, double* frames_host, int capacity, int ring_slots, int include_t0)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    if (capacity < 0 || ring_slots < 0) return fail(c, TDSE_EINVAL, "tdse_set_frame_stream: capacity, ring_slots must be >= 0");
    if (capacity > 0 && (!frames_host || ring_slots < 2)) return fail(c, TDSE_EINVAL, "tdse_set_frame_stream: needs a host buffer and at least 2 ring slots");
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    free_frame_stream(c);
    if (c->frames) { cudaFree(c->frames); c->frames = nullptr; c->max_frames = 0; }
    c->frames_t0 = include_t0 ? 1 : 0;
    if (capacity > 0) {
        ring_slots = std::min(ring_slots, capacity);
        cudaError_t e = cudaMalloc(&c->fs_ring, (size_t)ring_slots * c->g.batch * c->g.plane * sizeof(double));
        if (e != cudaSuccess) { cudaGetLastError(); c->fs_ring = nullptr; return fail(c, TDSE_ENOMEM, std::string("tdse_set_frame_stream: ring: ") + cudaGetErrorString(e)); }
        if ((e = cudaStreamCreateWithFlags(&c->fs_stream, cudaStreamNonBlocking)) != cudaSuccess) { free_frame_stream(c); return fail(c, TDSE_ECUDA, "tdse_set_frame_stream: stream"); }
        c->fs_written.assign(ring_slots, nullptr); c->fs_copied.assign(ring_slots, nullptr); c->fs_busy.assign(ring_slots, 0);
        for (int q = 0; q < ring_slots; ++q) {
            if (cudaEventCreateWithFlags(&c->fs_written[q], cudaEventDisableTiming) != cudaSuccess ||
                cudaEventCreateWithFlags(&c->fs_copied[q], cudaEventDisableTiming) != cudaSuccess) {
                free_frame_stream(c);
                return fail(c, TDSE_ECUDA, "tdse_set_frame_stream: events");
            }
        }
        c->fs_host = frames_host; c->fs_slots = ring_slots; c->fs_capacity = capacity;
        int max_pitch = 0;
        if (cudaDeviceGetAttribute(&max_pitch, cudaDevAttrMaxPitch, c->device) != cudaSuccess) { cudaGetLastError(); max_pitch = 0; }
        c->fs_copy2d = (size_t)capacity * c->g.plane * sizeof(double) <= (size_t)std::max(max_pitch, 0);
    }
    return reset_detector(c);
}

int tdse_frames_sync(tdse_ctx* c, int* nframes)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    if (!c->fs_ring) return fail(c, TDSE_ESTATE, "tdse_frames_sync: streamed frame mode is off (tdse_set_frame_stream)");
    CU_TRY(c, cudaStreamSynchronize(c->stream));       // every sample has been launched and has handed its slot over ...
    CU_TRY(c, cudaStreamSynchronize(c->fs_stream));    // ... and every copy has landed
    if (nframes) *nframes = std::min(c->nframes, c->fs_capacity);
    return TDSE_OK;
}

int tdse_dissimilarity(tdse_ctx* c, int first_frame, int last_frame, double* d_host)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    if (!d_host) return fail(c, TDSE_EINVAL, "tdse_dissimilarity: NULL");
    if (!c->frames) return fail(c, TDSE_ESTATE, "tdse_dissimilarity: frame mode is off (tdse_set_frames)");
    const int have = std::min(c->nframes, c->max_frames);
    if (first_frame < 0 || last_frame < first_frame || last_frame >= have)
        return fail(c, TDSE_EINVAL, "tdse_dissimilarity: frame window exceeds the frames kept");
    const int nwin = last_frame - first_frame + 1, batch = c->g.batch;
    int rc = ensure_partial(c, (size_t)batch * batch * nwin + (size_t)batch * batch);
    if (rc) return rc;
    double* inner = c->partial;
    double* d_dev = c->partial + (size_t)batch * batch * nwin;
    const int tiles = (batch + kDisTile - 1) / kDisTile;
    dissimilarity_inner_kernel<<<dim3((unsigned)(tiles * tiles), (unsigned)nwin), 256, 0, c->stream>>>(
        c->frames, batch, (long long)c->max_frames * c->g.plane, (int)c->g.plane, c->m.dx * c->m.dy, first_frame, nwin, inner);
    CU_LAUNCH_CHECK(c);
    dissimilarity_finish_kernel<<<(batch * batch + 127) / 128, 128, 0, c->stream>>>(inner, batch, nwin, d_dev);
    CU_LAUNCH_CHECK(c);
    CU_TRY(c, cudaMemcpyAsync(d_host, d_dev, (size_t)batch * batch * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    return TDSE_OK;
}

int tdse_detector_device(tdse_ctx* c, double** image_device, double** trace_device, int* max_samples)
{
    if (!c) return TDSE_EINVAL;
    if (image_device) *image_device = c->D;
    if (trace_device) *trace_device = c->trace;
    if (max_samples) *max_samples = c->max_samples;
    return TDSE_OK;
}

int tdse_read_psi(tdse_ctx* c, int b, void* R_host, void* I_host)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    if (b < 0 || b >= c->g.batch) return fail(c, TDSE_EINVAL, "tdse_read_psi: entry out of range");
    if (!c->ws || !c->have_state[b]) return fail(c, TDSE_ESTATE, "tdse_read_psi: state not set");
    int rc;
    if (R_host && (rc = copy_entry(c, entry_ptr(c, c->R[c->cur], b), R_host, cudaMemcpyDeviceToHost, false))) return rc;
    if (I_host && (rc = copy_entry(c, entry_ptr(c, c->I[c->cur], b), I_host, cudaMemcpyDeviceToHost, false))) return rc;
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    return TDSE_OK;
}

int tdse_read_potential(tdse_ctx* c, int b, void* V_host)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    if (b < 0 || b >= c->g.batch) return fail(c, TDSE_EINVAL, "tdse_read_potential: entry out of range");
    if (!c->ws || !c->have_V[b]) return fail(c, TDSE_ESTATE, "tdse_read_potential: potential not set");
    if (!V_host) return fail(c, TDSE_EINVAL, "tdse_read_potential: NULL");
    { int rc = copy_entry(c, entry_ptr(c, c->V, b), V_host, cudaMemcpyDeviceToHost, false); if (rc) return rc; }
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    return TDSE_OK;
}

int tdse_norm(tdse_ctx* c, int b, double* q_visscher, double* q_paper)
{
    if (!c) return TDSE_EINVAL;
    ENTER_DEVICE(c);
    if (b < 0 || b >= c->g.batch) return fail(c, TDSE_EINVAL, "tdse_norm: entry out of range");
    if (!c->ws || !c->have_state[b] || !c->have_V[b]) return fail(c, TDSE_ESTATE, "tdse_norm: potential and state must be set");
    const unsigned nblk = (unsigned)((c->g.cells + 255) / 256);
    int rc = ensure_partial(c, (size_t)2 * nblk);
    if (rc) return rc;
    if (c->dtype == TDSE_F32)
        norm_partial_kernel<float><<<nblk, 256, 0, c->stream>>>(c->g, c->m, (const float*)entry_ptr(c, c->V, b),
            (const float*)c->mask_dev, (const float*)entry_ptr(c, c->R[c->cur], b), (const float*)entry_ptr(c, c->I[c->cur], b), c->partial);
    else
        norm_partial_kernel<double><<<nblk, 256, 0, c->stream>>>(c->g, c->m, (const double*)entry_ptr(c, c->V, b),
            (const double*)c->mask_dev, (const double*)entry_ptr(c, c->R[c->cur], b), (const double*)entry_ptr(c, c->I[c->cur], b), c->partial);
    CU_LAUNCH_CHECK(c);
    reduce_rows_kernel<<<1, 256, 0, c->stream>>>(c->partial, (int)nblk, 2, c->m.dx * c->m.dy * c->m.dz, c->scalars);
    CU_LAUNCH_CHECK(c);
    double q[2];
    CU_TRY(c, cudaMemcpyAsync(q, c->scalars, sizeof q, cudaMemcpyDeviceToHost, c->stream));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    if (q_visscher) *q_visscher = q[0];
    if (q_paper) *q_paper = q[1];
    return TDSE_OK;
}

int tdse_set_option(tdse_ctx* c, const char* key, long long value)
{
    if (!c || !key) return TDSE_EINVAL;
    const std::string k(key);
    if (k == "kernel") {
        if (value < TDSE_KERNEL_AUTO || value > TDSE_KERNEL_FUSED) return fail(c, TDSE_EINVAL, "tdse_set_option: kernel");
        c->opt_kernel = (int)value;
    } else if (k == "tblock") {
        if (value < 0 || value > 2) return fail(c, TDSE_EINVAL, "tdse_set_option: tblock must be 0..2");
        c->opt_tblock = (int)value;
    } else if (k == "prefetch") {
        if (value < 0 || value > 4) return fail(c, TDSE_EINVAL, "tdse_set_option: prefetch must be 0..4");
        c->opt_pf = (int)value;
    } else if (k == "z_chunks") {
        if (value < 0) return fail(c, TDSE_EINVAL, "tdse_set_option: z_chunks must be >= 0");
        c->opt_chunks = (int)value;
    } else if (k == "variant") {
        if (value < 0 || value > 2) return fail(c, TDSE_EINVAL, "tdse_set_option: variant must be 0 (auto), 1 or 2");
        c->opt_variant = (int)value;
    } else if (k == "pdl") {
        c->opt_pdl = value ? 1 : 0;
    } else if (k == "allow_unstable") {
        c->allow_unstable = value ? 1 : 0;
    } else {
        return fail(c, TDSE_EINVAL, "tdse_set_option: unknown key " + k);
    }
    return TDSE_OK;
}

int tdse_get_info(const tdse_ctx* c, const char* key, long long* value)
{
    if (!c || !key || !value) return TDSE_EINVAL;
    const std::string k(key);
    if (k == "launches") *value = c->launches;
    else if (k == "steps") *value = c->steps;
    else if (k == "kernel") *value = c->last_kernel;
    else if (k == "tblock") *value = c->last_tblock;
    else if (k == "pingpong") *value = c->pingpong ? 1 : 0;
    else if (k == "tile_x") *value = c->last_tile_x;
    else if (k == "tile_y") *value = c->last_tile_y;
    else if (k == "z_chunks") *value = c->last_chunks;
    else if (k == "nsamples") *value = c->nsamples;
    else if (k == "nframes") *value = c->nframes;
    else return TDSE_EINVAL;
    return TDSE_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// tdse_dissimilarity_static: eq (16) without any allocation (include/tdse.h says who needs that and why).
// The scratch that tdse_dissimilarity takes from cudaMalloc is this fixed array instead.  It lives in the module
// image, so each GPU that loads the library carries it (2 MiB) until the process ends, and all calls on a GPU share it.
// ---------------------------------------------------------------------------------------------
static __device__ __align__(256) double g_static_scratch[TDSE_STATIC_SCRATCH_DOUBLES];

namespace {

// Device address of g_static_scratch on each GPU, filled in by the first call made with that GPU current.  In host
// code `g_static_scratch` is only a handle for the runtime's symbol table -- handing it to a kernel as if it were a
// pointer would make the kernel dereference a host address -- so the real address is asked for once per device
// (the array has a different address in every device's copy of the module) and kept here.
double* g_static_scratch_addr[kMaxDevices] = {};

int static_scratch_for_current_device(double** out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return fail(nullptr, TDSE_ECUDA, std::string("tdse_dissimilarity_static: cudaGetDevice: ") + cudaGetErrorString(e)
                                         + " (no CPU fallback)");
    }
    if (dev < 0 || dev >= kMaxDevices) return fail(nullptr, TDSE_EINVAL, "tdse_dissimilarity_static: device ordinal out of range");
    double* p = g_static_scratch_addr[dev];       // racing first calls would both store the same address
    if (!p) {
        e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_static_scratch);
        if (e != cudaSuccess || !p) {
            cudaGetLastError();
            return fail(nullptr, TDSE_ECUDA, std::string("tdse_dissimilarity_static: cudaGetSymbolAddress: ") + cudaGetErrorString(e));
        }
        g_static_scratch_addr[dev] = p;
    }
    *out = p;
    return TDSE_OK;
}

// true if p is device (or managed) memory that the current device `dev` owns
bool is_memory_of_device(const void* p, int dev)
{
    cudaPointerAttributes a{};
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    if (a.type == cudaMemoryTypeManaged) return true;
    return a.type == cudaMemoryTypeDevice && a.device == dev;
}

}  // namespace

extern "C" int tdse_dissimilarity_static(const double* frames_device, int batch, int frames_per_entry, int ny, int nx,
                                         double dA, int first_frame, int last_frame, double* d_device, void* cuda_stream)
{
    const char* who = "tdse_dissimilarity_static: ";
    if (!frames_device || !d_device) return fail(nullptr, TDSE_EINVAL, std::string(who) + "NULL");
    if (batch < 1 || frames_per_entry < 1 || ny < 1 || nx < 1 || !(dA > 0.0))
        return fail(nullptr, TDSE_EINVAL, std::string(who) + "batch, frames_per_entry, ny, nx must be >= 1 and dA > 0");
    if ((long long)ny * nx > std::numeric_limits<int>::max())
        return fail(nullptr, TDSE_EINVAL, std::string(who) + "ny*nx exceeds 2^31 - 1");
    if (first_frame < 0 || last_frame < first_frame || last_frame >= frames_per_entry)
        return fail(nullptr, TDSE_EINVAL, std::string(who) + "frame window outside [0, frames_per_entry)");
    const int nwin = last_frame - first_frame + 1;
    const long long need = (long long)batch * batch * nwin;
    if (nwin > 65535) return fail(nullptr, TDSE_EINVAL, std::string(who) + "more than 65535 frames in the window");
    if (need > (long long)TDSE_STATIC_SCRATCH_DOUBLES) {
        char msg[256];
        snprintf(msg, sizeof msg, "%sbatch*batch*frames = %lld exceeds the fixed scratch of %d doubles; shorten the window, "
                 "split the batch, or use tdse_dissimilarity (which allocates)", who, need, (int)TDSE_STATIC_SCRATCH_DOUBLES);
        return fail(nullptr, TDSE_EINVAL, msg);
    }
    double* inner = nullptr;
    const int rc = static_scratch_for_current_device(&inner);     // first call on this GPU: looks the address up
    if (rc) return rc;
    int dev = -1;
    cudaGetDevice(&dev);
    if (!is_memory_of_device(frames_device, dev) || !is_memory_of_device(d_device, dev))
        return fail(nullptr, TDSE_EINVAL, std::string(who) + "frames_device and d_device must be device memory of the current device");
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const int npix = ny * nx;
    const int tiles = (batch + kDisTile - 1) / kDisTile;
    // Same two kernels, launch shapes and summation order as tdse_dissimilarity.  The first writes every
    // inner[(k*batch + j)*nwin + s] with j >= k, the second reads exactly those: no element of the shared array is read
    // before this call has written it, whatever an earlier call left there.
    dissimilarity_inner_kernel<<<dim3((unsigned)(tiles * tiles), (unsigned)nwin), 256, 0, stream>>>(
        frames_device, batch, (long long)frames_per_entry * npix, npix, dA, first_frame, nwin, inner);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) {
        dissimilarity_finish_kernel<<<(batch * batch + 127) / 128, 128, 0, stream>>>(inner, batch, nwin, d_device);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) return fail(nullptr, TDSE_ECUDA, std::string(who) + "kernel launch: " + cudaGetErrorString(e));
    return TDSE_OK;
}
