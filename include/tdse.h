/* tdse.h -- C ABI of libtdse: the FDTD leapfrog hot path of arXiv 2401.07416 on one B200.
 *
 * What the library computes (citations are /root/reference/PAPER.md line + equation):
 *   - the split psi = psi_R + i psi_I on a rectangular mesh, eqs (5)-(7), PAPER.md:60-72;
 *   - the leapfrog recurrence eq (9) (I half-step) then eq (8) (R half-step), PAPER.md:74-87,
 *     with c = hbar dt / (2 m dx^2) and c_v = dt / hbar;
 *   - periodic wrap of neighbour indices, eqs (13)-(14), or zero-Dirichlet faces;
 *   - an absorbing layer (eq (10), realised as a multiplicative polynomial mask);
 *   - the Gaussian packet of eq (3), started on the staggered time grid;
 *   - the detector-plane density of eq (15), with the staggered density of PAPER.md:87;
 *   - a synthetic potential summed from an atom list (BASELINE.json north_star (1)), which stands in for
 *     the DFT potential of PAPER.md:50, 164.
 * DESIGN.md lists every reading taken where the paper is silent or garbled.
 *
 * Conventions
 *   - Every call returns an int status (TDSE_OK = 0, negative = error); nothing throws or aborts
 *     across this boundary; out-parameters are written only on success; tdse_last_error() gives text.
 *   - Layout: batch entry b, grid point (i, j, k) at position (i dx, j dx, k dx) lives at
 *     flat offset ((b*nz + k)*ny + j)*nx + i, x fastest, in the context's dtype (float or double).
 *     (The paper stores z fastest; this is a relabelling, reading 17.)
 *   - "host" / "device" in a parameter name says where the pointer must live.  The caller owns every
 *     buffer it passes in; the library copies atom lists before returning.  A workspace given to
 *     tdse_bind() stays owned by the caller and must outlive the context.
 *   - All work is enqueued on the stream given to tdse_bind() (default: the legacy null stream).
 *     tdse_step() is asynchronous; calls that return data to the host synchronise that stream.
 *   - One context is not thread-safe; distinct contexts are independent and may be driven from different host
 *     threads.  The context-free error slot (tdse_last_error(NULL): tdse_create failures, tdse_dissimilarity_static)
 *     is per host thread.  tdse_dissimilarity_static shares one scratch array per GPU across all callers (see there).
 *   - There is no CPU fallback: every call needs a CUDA device and fails with TDSE_ECUDA without one.
 */
#ifndef TDSE_H
#define TDSE_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tdse_ctx tdse_ctx;  /* opaque; created by tdse_create, freed by tdse_destroy */

enum { TDSE_F32 = 0, TDSE_F64 = 1 };
enum { TDSE_BC_PERIODIC = 0, TDSE_BC_DIRICHLET = 1 };  /* Dirichlet: values at index -1 and n are zero */
enum {
    TDSE_OK = 0,
    TDSE_EINVAL = -1,     /* bad argument */
    TDSE_ENOMEM = -2,     /* host or device allocation failed / workspace too small */
    TDSE_ECUDA = -3,      /* CUDA runtime error (text in tdse_last_error) */
    TDSE_ESTATE = -4,     /* call out of order (e.g. step before potential and state are set) */
    TDSE_EUNSTABLE = -5   /* dt above the sufficient stability bound, see tdse_step */
};

/* One atom of the synthetic potential.  screen <= 0 (or non-finite) means "unscreened". */
typedef struct { double x, y, z, Z, soft2, screen; } tdse_atom;

/* Kernel variants selectable with tdse_set_option("kernel", v). */
enum {
    TDSE_KERNEL_AUTO = 0,     /* fused where the shape allows it, else two-pass */
    TDSE_KERNEL_TWOPASS = 1,  /* one thread per cell, eq (9) launch then eq (8) launch, in place */
    TDSE_KERNEL_FUSED = 2     /* z-marching fused R+I kernel, T full steps per pass.  Needs the 5-array (ping-pong)
                               * workspace, nx*sizeof(element) a multiple of 16, even ny, nx >= 8, ny >= 8;
                               * tdse_step returns TDSE_EINVAL if it is forced on anything else. */
};

/* Create a context for `batch` independent nx*ny*nz grids with cubic cells of edge dx, time step dt,
 * particle mass `mass`, reduced Planck constant `hbar`, arithmetic/storage type `dtype`.
 * Defaults: periodic on all three axes, no absorber, detector off.
 * The context belongs to the CUDA device that is current in this call: every later call on it runs on that device
 * whatever device the caller has current then (and leaves the caller's device current on return); a workspace
 * passed to tdse_bind must live on it.
 * Errors: TDSE_EINVAL (sizes < 1, non-positive dx/dt/mass/hbar, unknown dtype), TDSE_ECUDA, TDSE_ENOMEM. */
int tdse_create(tdse_ctx** out, int nx, int ny, int nz, int batch,
                double dx, double dt, double mass, double hbar, int dtype);

/* Free the context and everything the library allocated.  NULL is accepted. */
int tdse_destroy(tdse_ctx* ctx);

/* Anisotropic mesh (c_x, c_y, c_z = hbar dt / (2 m dx^2), ... ; the paper's own mesh is
 * 35.4/240 x 40.9/240 x 70/420 Angstrom).  tdse_create makes cubic cells (dy = dz = dx); this call
 * changes the spacing along y and z.  Grid point (i, j, k) sits at (i dx, j dy, k dz); the trace carries dx*dy, the
 * norms dx*dy*dz.  Potential and state must be set again afterwards (TDSE_ESTATE from tdse_step otherwise).
 * Errors: TDSE_EINVAL. */
int tdse_set_spacing(tdse_ctx* ctx, double dy, double dz);

/* Bytes of device workspace for the R, I, V grids (pingpong = 0: 3 arrays, two-pass kernels only;
 * pingpong = 1: 5 arrays, needed by the fused kernels).  Inside the workspace every xy plane is stored
 * with a frame of 4 columns and 4 rows on each side (periodic images or Dirichlet zeros, which lets the
 * fused kernel fetch tile + halo with one TMA box): one array holds batch*nz*(ny+8)*(nx+8) elements,
 * rounded up to 256 bytes.  The layout is private to the library; every buffer that crosses this ABI
 * is the plain [z][y][x] grid.  Returns 0 on invalid arguments. */
size_t tdse_workspace_bytes(int nx, int ny, int nz, int batch, int dtype, int pingpong);

/* Use caller-owned device memory (e.g. a torch tensor) and a caller-owned CUDA stream (a cudaStream_t
 * passed as void*; NULL = legacy default stream).  `bytes` >= tdse_workspace_bytes(..., 0); if it is
 * also >= tdse_workspace_bytes(..., 1) the fused kernels become available.  dev_workspace must be
 * 256-byte aligned.  If tdse_bind is never called the library allocates its own 5-array workspace on
 * first use.  Rebinding discards potential and state.  Errors: TDSE_EINVAL, TDSE_ENOMEM. */
int tdse_bind(tdse_ctx* ctx, void* dev_workspace, size_t bytes, void* cuda_stream);

/* Boundary condition per axis and the absorbing layers at the two z faces.
 * The freshly updated field is multiplied by M[k] after each half-step, with
 *   M[k] = 1 - strength * xi^power,  xi = (absorb_lo - k)/absorb_lo  for k < absorb_lo,
 *                                    xi = (k - (nz-1-absorb_hi))/absorb_hi  for k > nz-1-absorb_hi,
 * M = 1 elsewhere; 0 cells = that layer is off.  Errors: TDSE_EINVAL (unknown bc, negative widths,
 * absorb_lo + absorb_hi > nz, strength outside [0, 1], power < 1).
 * May be called before or after potential and state are loaded: when an x or y flag changes, the private storage
 * frames (tdse_workspace_bytes) of the data already loaded are rewritten for the new flags. */
int tdse_set_boundary(tdse_ctx* ctx, int bcx, int bcy, int bcz,
                      int absorb_lo, int absorb_hi, double strength, int power);

/* Build V for entry b (b = -1: all entries) on the device from `natoms` atoms in HOST memory:
 *   V = min(max( sum_a -Z_a * exp(-r_a/screen_a) / sqrt(r_a^2 + soft2_a), vmin), vmax)
 * r_a = distance from the grid point to atom a, nearest periodic image on periodic axes, true distance
 * on Dirichlet axes; rcut > 0 skips atoms with r_a > rcut.  Accumulated in double in list order and
 * rounded once to the context dtype.  Uses the boundary flags in force at the time of the call.
 * Errors: TDSE_EINVAL (b out of range, natoms < 0, NULL with natoms > 0, vmin > vmax), TDSE_ECUDA. */
int tdse_set_potential(tdse_ctx* ctx, int b, const tdse_atom* atoms_host, int natoms,
                       double vmin, double vmax, double rcut);

/* Same, with the atom list already in DEVICE memory (must stay valid until the stream reaches the
 * build kernel; the library does not copy it). */
int tdse_set_potential_device(tdse_ctx* ctx, int b, const tdse_atom* atoms_device, int natoms,
                              double vmin, double vmax, double rcut);

/* Build V for every entry in ONE launch (BASELINE.json north_star (4): many independent configurations, e.g. the
 * paper's 879 thin-film structures): entry e uses atoms[offsets_host[e] .. offsets_host[e+1]) of one
 * concatenated list.  `offsets_host` is a HOST array of batch+1 non-decreasing ints; `atoms` is in host memory
 * (on_device = 0) or in device memory (on_device = 1, not copied: must stay valid until the stream reaches the build
 * kernel).  Same definition and summation order as tdse_set_potential.  Atoms that every list starts with (a shared
 * substrate) are found by the library (bitwise comparison) and summed once: a cell's sum then starts from the
 * shared partial sum, which is the same sequence of operations as the plain list-order sum, so the result does not
 * depend on it.  With on_device = 1 and batch >= 2 the call synchronises the stream once (one int comes back).
 * Errors: TDSE_EINVAL (NULL, decreasing offsets, vmin > vmax), TDSE_ENOMEM, TDSE_ECUDA. */
int tdse_set_potential_batch(tdse_ctx* ctx, const tdse_atom* atoms, const int* offsets_host, int on_device,
                             double vmin, double vmax, double rcut);

/* Potential from a unit-cell grid (PAPER.md:148, 213 step (ii): "expansion and interpolation of the electrostatic
 * potential onto the mesh points"; the paper spends 15 min per configuration on the host here).  cell: mz*my*mx
 * doubles, [z][y][x], HOST (on_device = 0) or DEVICE (on_device = 1), samples at spacings (ax/mx, ay/my,
 * az/(mz-1)).  The cell repeats periodically in x and y (the slab's supercell); below z0 and above z0 + az the
 * nearest z plane is used.  V at mesh point (i dx, j dy, k dz) is the trilinear interpolation at
 * (i dx - x0, j dy - y0, k dz - z0), clamped to [vmin, vmax], rounded once to the context dtype (DESIGN.md
 * reading 24).  b = -1: all entries.  The stability check uses max(|vmin|, |vmax|).  Errors: TDSE_EINVAL, TDSE_ECUDA. */
int tdse_set_potential_cell(tdse_ctx* ctx, int b, const double* cell, int on_device, int mx, int my, int mz,
                            double ax, double ay, double az, double x0, double y0, double z0, double vmin, double vmax);

/* Raw potential grid for entry b (b = -1: the same grid for all entries), nx*ny*nz values of the
 * context dtype, layout [z][y][x]; on_device says where V lives (a gridded V). */
int tdse_set_potential_grid(tdse_ctx* ctx, int b, const void* V, int on_device);

/* Gaussian packet, eq (3) PAPER.md:52 with a signed wave vector:
 *   psi0 = A exp(-|r - r0|^2 / (2 sigma^2)) exp(+i k.(r - r0)),  A = amplitude, or (pi sigma^2)^(-3/4)
 * when amplitude == 0.  The paper's case is k = (0, 0, -2 pi / lambda), eq (4).  Stores
 *   R^0 = Re psi0,   I^{-1/2} = Im psi0 + (1/2) (dt/hbar) (H Re psi0)
 * (staggered start, reading 4), evaluated in double from the stored V and rounded once.
 * Resets the step counter and the detector.  b = -1: all entries.
 * Errors: TDSE_ESTATE (potential of that entry not set), TDSE_EINVAL (sigma <= 0, b out of range). */
int tdse_set_wavepacket(tdse_ctx* ctx, int b, double x0, double y0, double z0, double sigma,
                        double kx, double ky, double kz, double amplitude);

/* Raw state for entry b (b = -1: the same state for all entries): R^n and I^{n-1/2}, nx*ny*nz values
 * each of the context dtype, [z][y][x].  Resets the step counter and the detector: this is a fresh start from a given
 * wavefunction, not a checkpoint restore -- the sampling phase, the accumulated image, the trace and the frames begin
 * again at zero, so a caller that resumes a run keeps its own copy of those and adds to it. */
int tdse_set_state(tdse_ctx* ctx, int b, const void* R, const void* I_half, int on_device);

/* Detector plane k_plane (0 <= k_plane < nz), sampled after every `every`-th full step counted from the
 * last reset (eq (15), h = `every`); every = 0 switches it off.  Each sample adds
 *   rho(i,j) = R^s(i,j,k)^2 + I^{s-1/2}(i,j,k)^2      (density of PAPER.md:87)
 * to a per-entry image (double) and appends dx^2 * sum_ij rho to a per-entry trace.  Resets image,
 * trace and step counter.  `max_samples` traces are kept per entry (further samples still accumulate
 * into the image but are not recorded in the trace).  The trace buffer is kept (and its device pointer stays
 * valid) while `max_samples` does not change; with the same `max_samples` the call does not synchronise.
 * Errors: TDSE_EINVAL; TDSE_ENOMEM (the previous detector set-up is still in force). */
int tdse_set_detector(tdse_ctx* ctx, int k_plane, int every, int max_samples);

/* Advance every entry by n full time steps (eq (9) then eq (8), mask, detector), asynchronously on the
 * bound stream.  Errors: TDSE_ESTATE if any entry lacks potential or state; TDSE_EUNSTABLE if
 * dt > 2 hbar / (12 hbar^2 / (2 m dx^2) + max|V|) (sufficient bound for max|eig(dt H / hbar)| < 2;
 * max|V| is taken over the clamp limits / raw grids seen so far), unless option "allow_unstable" is 1. */
int tdse_step(tdse_ctx* ctx, int n);

/* Copy entry b's accumulated detector image (ny*nx doubles, [y][x]) and the first min(cap, nsamples)
 * trace values to HOST memory; *nsamples = samples taken so far.  NULL pointers skip that output.
 * Synchronises the stream. */
int tdse_detector_read(tdse_ctx* ctx, int b, double* image_host, double* trace_host, int cap, int* nsamples);

/* Frame mode (eq (15): the paper's product is the trajectory rho = {rho(0), rho(h dt), ...} of
 * detector-plane densities).  With max_frames > 0 every detector sample also keeps its frame
 * rho_s[j][i] = (R^s)^2 + (I^{s-1/2})^2 in a device buffer [batch][max_frames][ny][nx] (double); with include_t0 != 0
 * frame 0 is rho at s = 0, taken from the state in memory when tdse_step is first called, and sample s*every is
 * frame s (else sample s*every is frame s-1).  Samples beyond max_frames are counted but not kept.  max_frames = 0
 * turns frame mode off.  Resets image, trace, frame and step counters.  Errors: TDSE_EINVAL, TDSE_ENOMEM. */
int tdse_set_frames(tdse_ctx* ctx, int max_frames, int include_t0);

/* Copy frames first .. first+count-1 of entry b to frames_host (HOST, count*ny*nx doubles, [frame][y][x]);
 * *nframes (may be NULL) receives the number of frames taken so far.  Synchronises.
 * Errors: TDSE_EINVAL (entry or frame range). */
int tdse_frames_read(tdse_ctx* ctx, int b, int first, int count, double* frames_host, int* nframes);

/* Device pointer of the frame buffer (library-owned; valid until tdse_set_frames / tdse_destroy). */
int tdse_frames_device(tdse_ctx* ctx, double** frames_device, int* max_frames, int* nframes);

/* Streamed frame mode (a 5000-step run keeps 250 frames per configuration, 879 configurations): the same
 * frames as tdse_set_frames, but the device holds only a ring of `ring_slots` (>= 2) sample slots [slot][batch][ny][nx]; as
 * soon as a sample's slot is written it is copied (one asynchronous strided copy per slot, on a second stream owned by
 * the library) into `frames_host`, a HOST buffer of batch * capacity * ny * nx doubles laid out [batch][capacity][ny][nx]
 * (page-locked memory lets the copies overlap the stepping; pageable memory works but serialises).  The stepping stream
 * waits only when it comes back to a slot whose copy has not left yet.  Frames beyond `capacity` are dropped.  The buffer
 * belongs to the caller and must stay valid until tdse_frames_sync has returned after the last step (or the mode is
 * switched off with capacity = 0).  Excludes tdse_set_frames / tdse_dissimilarity (which need the frames on the device).
 * Resets the detector.  When capacity * ny * nx * 8 bytes exceeds the device's 2-D copy pitch limit (cudaDevAttrMaxPitch,
 * 2^31 - 1 bytes) a slot leaves as one copy per entry instead of one strided copy; the result is the same.
 * Errors: TDSE_EINVAL, TDSE_ENOMEM, TDSE_ECUDA. */
int tdse_set_frame_stream(tdse_ctx* ctx, double* frames_host, int capacity, int ring_slots, int include_t0);

/* Wait until every frame sampled so far has landed in the host buffer of tdse_set_frame_stream; *nframes = frames kept per
 * entry.  Errors: TDSE_ESTATE if the streamed mode is off. */
int tdse_frames_sync(tdse_ctx* ctx, int* nframes);

/* Pairwise dissimilarity of the batch entries' trajectories, eq (16) PAPER.md:219-221:
 *   d_kj = 1/(t1-t0) int_{t0}^{t1} ( int_D (rho_k - rho_j)^2 dr )^{1/2} dt
 * evaluated as the mean over frames first_frame .. last_frame (inclusive) of sqrt(dx^2 * sum over the plane of
 * (rho_k - rho_j)^2) (reading 23).  d_host: HOST, batch*batch doubles, symmetric, zero diagonal.
 * Synchronises.  Errors: TDSE_ESTATE (frame mode off), TDSE_EINVAL (window exceeds the frames kept). */
int tdse_dissimilarity(tdse_ctx* ctx, int first_frame, int last_frame, double* d_host);

/* Eq (16) for callers that must not allocate GPU memory.
 *
 * Who this is for.  tdse_dissimilarity() sizes a per-context reduction buffer with cudaMalloc the first time it sees a
 * new batch x window.  Some programs cannot let a library do that: a job that has handed (nearly) all of the 180 GB to
 * the grids, as the fill-HBM configuration does, has nothing left for cudaMalloc to find; a host whose device memory
 * is owned by one pool (an inference server, a torch caching allocator with a hard cap) treats a side allocation as a
 * budget violation or an out-of-memory risk; and cudaMalloc/cudaFree stall the whole device, which a loop that is
 * stepping other contexts on other streams cannot afford.  This call does the same computation with the same kernels
 * and never calls cudaMalloc, cudaFree or any other allocating routine.
 *
 * How.  The per-(pair, frame) partial results go to a fixed array of TDSE_STATIC_SCRATCH_DOUBLES doubles (2 MiB) that
 * is part of the library image: every GPU that loads libtdse holds those 2 MiB from load until the process exits,
 * whether or not this call is ever made.  Inputs and outputs stay the caller's:
 *   frames_device  DEVICE, [batch][frames_per_entry][ny][nx] doubles (the layout tdse_frames_device returns), read only
 *   d_device       DEVICE, batch*batch doubles, written: symmetric, zero diagonal, same values as tdse_dissimilarity
 *   dA             area of one detector pixel (dx*dy)
 *   cuda_stream    a cudaStream_t passed as void* (NULL = legacy default stream); the work is enqueued there and the
 *                  call returns without synchronising -- d_device is ready when that stream reaches this point.
 * Both pointers must belong to the device that is current in the calling thread.
 *
 * Limit: batch*batch*(last_frame-first_frame+1) <= TDSE_STATIC_SCRATCH_DOUBLES (e.g. 32 trajectories x the paper's 250
 * frames); anything larger is refused with TDSE_EINVAL and a message, nothing is launched.
 *
 * Sharing.  There is one array per GPU and every call on that GPU uses it.  A call overwrites each element it later
 * reads, so nothing has to be cleared and what the previous call left behind is never seen.  Two calls that can be in
 * flight on the same GPU at once (different streams, or two host threads) race on the array and both results are
 * garbage: put them on one stream, or order them with events.
 *
 * First call.  The first call on each GPU looks up the array's device address (cudaGetSymbolAddress, which may also
 * make the CUDA runtime load the module); later calls reuse it.  Make that first call during set-up, before starting
 * any stream capture on that GPU.
 *
 * Errors: TDSE_EINVAL (NULL, sizes < 1, bad window, over the limit, pointer not device memory of the current
 * device), TDSE_ECUDA.  Text goes to the global slot: tdse_last_error(NULL). */
enum { TDSE_STATIC_SCRATCH_DOUBLES = 262144 };
int tdse_dissimilarity_static(const double* frames_device, int batch, int frames_per_entry, int ny, int nx, double dA,
                              int first_frame, int last_frame, double* d_device, void* cuda_stream);

/* Device pointers to the detector image [batch][ny][nx] and trace [batch][max_samples] (doubles);
 * valid until the next tdse_set_detector or tdse_destroy.  Does not synchronise. */
int tdse_detector_device(tdse_ctx* ctx, double** image_device, double** trace_device, int* max_samples);

/* Copy entry b's R^n and I^{n-1/2} ([z][y][x], context dtype) to HOST memory. Synchronises. */
int tdse_read_psi(tdse_ctx* ctx, int b, void* R_host, void* I_host);

/* Copy entry b's potential ([z][y][x], context dtype) to HOST memory. Synchronises. */
int tdse_read_potential(tdse_ctx* ctx, int b, void* V_host);

/* Diagnostics for entry b, accumulated in double:
 *   q_paper    = dx^3 sum (R^n)^2 + (I^{n-1/2})^2
 *   q_visscher = dx^3 sum (R^n)^2 + I^{n+1/2} I^{n-1/2}         (conserved exactly when M == 1)
 * I^{n+1/2} is one look-ahead eq (9) half-step (with mask) evaluated in double; state is not modified.
 * Either pointer may be NULL.  Synchronises. */
int tdse_norm(tdse_ctx* ctx, int b, double* q_visscher, double* q_paper);

/* Options: "kernel" (TDSE_KERNEL_*), "tblock" (full steps fused per pass, 0 = auto, 1..2),
 * "prefetch" (planes the fused kernel keeps in flight through TMA, 0 = deepest that fits, 1..4),
 * "z_chunks" (z chunks per tile column in the fused launch, 0 = chosen by the launcher),
 * "pdl" (0/1, default 1: fused launches carry the programmatic-stream-serialization attribute, so the next
 * launch becomes resident while the previous one drains; results are bit-identical either way),
 * "variant" (0 = the launcher decides, 1 / 2 = force on / off the fused kernel whose per-plane block barrier is a split
 * arrive / wait mbarrier; same arithmetic in the same order, so results are bit-identical),
 * "allow_unstable" (0/1).  Errors: TDSE_EINVAL for unknown keys or values. */
int tdse_set_option(tdse_ctx* ctx, const char* key, long long value);

/* Introspection: "launches" (kernels launched by this context so far), "steps" (full steps since the last
 * reset), "kernel" / "tblock" (what tdse_step used last), "pingpong" (1 if 5-array workspace),
 * "tile_x", "tile_y", "z_chunks" (fused launch shape used last), "nsamples" (detector samples taken since the last
 * reset), "nframes" (frames taken since the last reset, kept or not).  Errors: TDSE_EINVAL. */
int tdse_get_info(const tdse_ctx* ctx, const char* key, long long* value);

/* Text of the last error on this context ("" if none).  Never NULL.  ctx may be NULL (global slot used
 * by tdse_create failures). */
const char* tdse_last_error(const tdse_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* TDSE_H */
