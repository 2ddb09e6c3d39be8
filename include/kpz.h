/* kpz.h -- C ABI of the B200-native octahedron-KPZ hot path (libkpz_b200.so).
 *
 * Method: Kelling & Odor, "Extremely large scale simulation of a Kardar-Parisi-Zhang model using graphics
 * cards", arXiv:1110.6745 (PAPER.md; "P:n" = PAPER.md line n).  The library advances a periodic L x L lattice of
 * slopes sigma_x, sigma_y in {+-1} (2 bits per site) by stochastic generalized-Kawasaki updates (eq. 2,
 * P:26-30) under the deterministic domain-decomposed random-sequential schedule of DESIGN.md section "Schedule"
 * (random origin per MCS in multiples of 4 sites; 4 tile colours in random order; T*T sequential
 * attempts per tile; every random number from Philox4x32-10 keyed by (seed; call, tile, MCS, replica)), and
 * reduces heights (eq. 3) to sum h, sum h^2 and the squared width W^2 (eq. 4).
 *
 * Conventions
 *   - All functions return an int32_t status: KPZ_OK (0) or a negative KPZ_E* code.  Nothing throws or aborts.
 *     kpz_last_error(ctx) returns a NUL-terminated message owned by the handle (valid until the next call on it).
 *   - "host" / "device" is stated for every pointer.  The caller owns every buffer it passes; the library owns
 *     only the opaque handle (freed by kpz_destroy) and small temporaries it allocates inside diagnostic calls.
 *   - Device buffers are allocated by the caller (PyTorch in the Python binding) and bound with kpz_bind; they
 *     must outlive the handle or be re-bound.  All work is enqueued on the bound CUDA stream.
 *   - A handle is not thread-safe; distinct handles are independent.
 *   - Coordinates are 0-based, x fastest: host slope arrays are row-major [y*L + x], values +1 / -1, with
 *     sigma_x(x,y) = h(x,y) - h(x-1,y) and sigma_y(x,y) = h(x,y) - h(x,y-1) (indices mod L, R3).
 *   - There is no CPU fallback: without a CUDA device every call that needs one returns KPZ_ECUDA.
 *
 * Device layout of the lattice buffer, per replica r at byte offset
 * r * L*L/4:  plane X = sigma_x followed by plane Y = sigma_y, each as L bit-lines, one per ROW y
 * (32-bit words, sigma(x,y) = bit (x & 31) of word y*(L/32) + (x >> 5)).  Bit 1 <=> sigma = +1.
 */
#ifndef KPZ_B200_H
#define KPZ_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define KPZ_OK 0
#define KPZ_EINVAL (-1)    /* bad argument (size, tile, probability, NULL pointer, replica out of range) */
#define KPZ_ENOMEM (-2)    /* a bound buffer is too small / temporary allocation failed */
#define KPZ_ECUDA (-3)     /* CUDA runtime error or no device; message in kpz_last_error */
#define KPZ_EOVERFLOW (-4) /* a requested int64 output does not fit (kpz_measure) */
#define KPZ_ESTATE (-5)    /* call order (not bound) or an invalid lattice state (kpz_set_slopes) */

typedef struct kpz_ctx kpz_ctx;

/* Sizes of the two device buffers kpz_bind expects, in bytes (host out-pointers).
 * lattice = n_replicas * L*L/4 (2 bits per site).  scratch holds per-replica counters and the partial
 * sums of the measurement kernels.  Same argument rules as kpz_create_batch; KPZ_EINVAL otherwise. */
int32_t kpz_workspace_bytes(uint32_t L, uint32_t tile, uint32_t n_replicas, size_t* lattice_bytes,
                            size_t* scratch_bytes);

/* Creates a handle for one lattice (north star signature kpz_create(L, p, q, tile, seed)).
 *   L    : linear size; a multiple of 2*tile and of 32.
 *   p, q : deposition / removal probabilities of eq. 2, each in [0,1]; accept iff a 32-bit Philox word
 *          is < floor(prob * 2^32) (always for prob = 1).
 *   tile : tile edge T, one of 4, 8, 16, 32, 64 (a power of two >= 4, multiples-of-4 offsets).
 *   seed : 64-bit Philox key.
 * *out receives the handle (host pointer).  Errors: KPZ_EINVAL, KPZ_ECUDA (no device). */
int32_t kpz_create(kpz_ctx** out, uint32_t L, double p, double q, uint32_t tile, uint64_t seed);

/* As kpz_create, for n_replicas >= 1 independent lattices ("independent runs") advanced together.
 * Replica r uses Philox counter word c3 = r; kpz_create == kpz_create_batch(..., 1). */
int32_t kpz_create_batch(kpz_ctx** out, uint32_t L, double p, double q, uint32_t tile, uint64_t seed,
                         uint32_t n_replicas);

/* Binds caller-owned DEVICE buffers (sizes from kpz_workspace_bytes; 16-byte aligned) and a CUDA stream
 * (cudaStream_t passed as void*, NULL = default stream).  Zeroes the scratch counters (asynchronously).
 * The lattice content is left as is.  lattice_bytes / scratch_bytes are the sizes the caller allocated;
 * KPZ_ENOMEM if too small. */
int32_t kpz_bind(kpz_ctx* ctx, void* d_lattice, size_t lattice_bytes, void* d_scratch, size_t scratch_bytes,
                 void* cuda_stream);

/* Flat zig-zag start of P:88: h(x,y) = (x+y) mod 2, i.e. sigma_x = sigma_y = +1 if (x+y) odd else -1;
 * W^2 = 1/4.  Resets h(0,0) = 0, the MCS clock and all counters of every replica.  Asynchronous. */
int32_t kpz_init_flat(kpz_ctx* ctx);

/* Advances every replica by `mcs` Monte Carlo steps (each exactly L*L attempts; 4 kernel launches per MCS on the
 * tiled path, one launch per call on the lattice-resident path, see kpz_set_path).
 * Asynchronous on the bound stream.  kpz_run(a); kpz_run(b) == kpz_run(a+b).  KPZ_EINVAL if the MCS clock
 * would pass 2^32 - 1 (it is a 32-bit Philox counter word). */
int32_t kpz_run(kpz_ctx* ctx, uint64_t mcs);

/* Chooses the kernels kpz_run uses; the results are bit-identical on every path:
 *   KPZ_PATH_AUTO (default): the lattice-resident kernel when the packed lattice fits in shared memory (L <= 512),
 *     the schedule is S4, with or without sub-sweeps (S6), without Poissonised counts, and the handle is small enough to
 *     be bound by launches and tile staging; else the tiled kernel;
 *   KPZ_PATH_TILED: kpz_update_kernel, one launch per colour pass (4 per MCS), any valid L;
 *   KPZ_PATH_RESIDENT: force the resident kernel (one launch per kpz_run call, the lattices of a CTA's replicas
 *     stay in shared memory for all MCS of the call); kpz_run then returns KPZ_EINVAL when the lattice or the
 *     schedule does not allow it.
 * KPZ_EINVAL for any other value. */
#define KPZ_PATH_AUTO 0
#define KPZ_PATH_TILED 1
#define KPZ_PATH_RESIDENT 2
int32_t kpz_set_path(kpz_ctx* ctx, int32_t path);

/* Chooses the domain-decomposition schedule for subsequent kpz_run calls:
 *   KPZ_SCHEDULE_COLOURS (default): S4 -- four tile colours in random order, halo write-back, exactly L*L effective
 *     attempts per MCS, 4 kernel launches per MCS;
 *   KPZ_SCHEDULE_DEAD_BORDER: S5 -- the paper's own device-level scheme: every tile in one pass (1 launch
 *     per MCS), attempts on the +x / +y edge sites of a tile do nothing ("dead borders"; a fraction 1 - (1-1/T)^2 of
 *     the L*L attempts), same origin shift and the same Philox streams.
 * May be called at any time between runs; KPZ_EINVAL for any other value. */
#define KPZ_SCHEDULE_COLOURS 0
#define KPZ_SCHEDULE_DEAD_BORDER 1
int32_t kpz_set_schedule(kpz_ctx* ctx, int32_t schedule);

/* Bias-reduction knob (S6): K sub-sweeps per MCS.  Sub-sweep j = 0..K-1 draws its own origin
 * shift and colour order (global draw with counter word c0 = j) and executes steps [j T^2/K, (j+1) T^2/K) of every
 * tile's Philox stream; K = 1 (default) is the schedule S4 / S5 itself.  An MCS stays exactly L*L attempts and costs
 * K times the launches and the tile staging.  K must divide tile*tile/8 (KPZ_EINVAL otherwise). */
int32_t kpz_set_sub_sweeps(kpz_ctx* ctx, uint32_t K);

/* Second bias-reduction knob (S7): Poissonised number of steps per tile and sub-sweep.  With
 * on != 0 every tile runs n steps of its stream, n drawn from the (integer-defined) Poisson law of mean
 * lambda = tile*tile/K with one Philox word per tile and sub-sweep, instead of exactly lambda steps -- the count
 * statistics of true random-sequential dynamics.  An MCS is then L*L attempts only on average; kpz_counters reports
 * the attempts really made.  Needs bound buffers (the table lives in the scratch buffer).  Synchronises. */
int32_t kpz_set_poisson(kpz_ctx* ctx, int32_t on);

/* Height reconstruction (eq. 3) and width (eq. 4).  HOST out-arrays of length n_replicas (any may be NULL).
 * sum_h, sum_h2: exact sums over all sites of h and h^2 with absolute heights anchored by h(0,0) (tracked:
 * 0 at kpz_init_flat, +-2 per accepted flip at site (0,0)).  W2 = (N*sum_h2 - sum_h^2)/N^2, N = L*L, from
 * 128-bit integers: one conversion to double, one division by (double)N^2.  Synchronises the stream.
 * Does not modify the lattice.  KPZ_EOVERFLOW if a requested sum does not fit int64 (W2 is still written). */
int32_t kpz_measure(kpz_ctx* ctx, int64_t* sum_h, int64_t* sum_h2, double* W2);

/* kpz_measure WITHOUT any allocation and without a host synchronisation, for callers that cannot allocate (code under
 * CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): the partial sums of the measurement
 * kernels live in a file-scope static device array of the library (819 456 bytes, held by every GPU that loads the
 * library until exit) instead of the bound scratch buffer.  LIMIT: L <= 8192 (KPZ_STATIC_MAX_L; the paper's largest
 * steady-state size); a larger handle gets KPZ_EINVAL and must use kpz_measure.
 *   replica : which lattice of the handle (input: the handle's bound lattice and its tracked h(0,0), both on the device)
 *   d_out   : caller-owned DEVICE buffer of 8 x 8 bytes, 8-byte aligned (output), written asynchronously on the bound
 *             stream: [0..3] the four 64-bit half-accumulators (lo / hi of sum (h - h00), lo / hi of sum (h - h00)^2:
 *             what kpz_slab_finalize takes), [4] sum h (int64), [5] sum h^2 (int64), [6] W^2 (double, the same
 *             128-bit integer arithmetic as kpz_measure: identical bits), [7] 1 if a sum does not fit int64 (it is
 *             then written as 0), else 0.
 * Calls no cudaMalloc, cudaFree or allocating routine; enqueues one 32-byte memset and four kernels.  The first call on
 * a device looks the array's address up (cudaGetSymbolAddress): make one call outside a graph capture first.
 * ALL handles and calls of a process share the one array per device, and it keeps the last call's contents (the call
 * clears what must start at zero): calls that may overlap on the GPU -- different streams, or graphs launched
 * concurrently -- RACE; serialise them (one stream, or events).  Does not modify the lattice or the handle's state.
 * Errors: KPZ_ESTATE (not bound, slab handle), KPZ_EINVAL (replica, d_out NULL / misaligned, L > 8192), KPZ_ECUDA. */
#define KPZ_STATIC_MAX_L 8192
int32_t kpz_measure_static(kpz_ctx* ctx, uint32_t replica, void* d_out);

/* Sampling-time driver ("the program calculates and writes out the width" at the times t_i of eq. 8):
 * advances to each absolute MCS clock times[i] (HOST array, strictly increasing, times[0] >= the current clock)
 * and measures there.  HOST out-arrays of n_times * n_replicas entries, sample-major [i * n_replicas + r] (any may
 * be NULL).  Equivalent to the kpz_run / kpz_measure calls it makes; returns KPZ_EOVERFLOW if any sample's int64
 * sum overflowed (W2 still written), KPZ_EINVAL for a bad time list. */
int32_t kpz_run_sampled(kpz_ctx* ctx, const uint64_t* times, uint32_t n_times, int64_t* sum_h, int64_t* sum_h2,
                        double* W2);

/* Frees the handle (not the bound buffers).  NULL is a no-op. */
int32_t kpz_destroy(kpz_ctx* ctx);

/* Waits for all work enqueued on the bound stream. */
int32_t kpz_synchronize(kpz_ctx* ctx);

const char* kpz_last_error(const kpz_ctx* ctx);

/* ---- parity / diagnostic / checkpoint extensions --------------------------------------------------------- */

/* Unpacks replica `replica` into HOST arrays sx, sy (int8, L*L each, row-major [y*L+x], values +-1).
 * Synchronises.  Allocates 2*L*L bytes of temporary device memory (KPZ_ENOMEM if that fails). */
int32_t kpz_get_slopes(kpz_ctx* ctx, uint32_t replica, int8_t* sx, int8_t* sy);

/* As kpz_get_slopes for the w x h window with lower-left site (x0, y0), periodic wrap; out arrays [j*w + i]. */
int32_t kpz_get_window(kpz_ctx* ctx, uint32_t replica, uint32_t x0, uint32_t y0, uint32_t w, uint32_t h,
                       int8_t* sx, int8_t* sy);

/* Packs HOST arrays (values must be +-1, else KPZ_EINVAL; the state must be curl-free with zero tilt --
 * sx(x+1,y)+sy(x+1,y+1) = sy(x,y+1)+sx(x+1,y+1), every row sum of sx and column sum of sy zero -- else
 * KPZ_ESTATE and the replica is left unchanged) into replica `replica`, and sets its h(0,0) to h00.
 * Does not touch the MCS clock or the flip counters.  Synchronises. */
int32_t kpz_set_slopes(kpz_ctx* ctx, uint32_t replica, const int8_t* sx, const int8_t* sy, int64_t h00);

/* Order-independent 64-bit hash of replica's state: sum over sites n = y*L+x of
 * bit_x(n)*mix64(2n) + bit_y(n)*mix64(2n+1) mod 2^64, bit = (sigma+1)/2, mix64 = splitmix64 finaliser
 * (z += 0x9E3779B97F4A7C15; z = (z^(z>>30))*0xBF58476D1CE4E5B9; z = (z^(z>>27))*0x94D049BB133111EB; z^(z>>31)).
 * HOST out-pointer.  Synchronises. */
int32_t kpz_state_hash(kpz_ctx* ctx, uint32_t replica, uint64_t* out);

/* Per-replica counters since kpz_init_flat (HOST out-pointers, any may be NULL): attempted updates
 * (= mcs * L*L unless S7 was on), accepted depositions and removals, tracked height of site (0,0), completed MCS.  Synchronises. */
int32_t kpz_counters(kpz_ctx* ctx, uint32_t replica, uint64_t* attempts, uint64_t* deposits, uint64_t* removals,
                     int64_t* h00, uint64_t* mcs);

/* Checkpoint: copies the packed lattice of ALL replicas (device layout above, kpz_workspace_bytes'
 * lattice_bytes bytes) between the bound device buffer and a HOST buffer (pinned memory makes the copy
 * asynchronous-capable; the calls synchronise before returning).  kpz_import_packed also takes the state the
 * lattice does not carry: per-replica h(0,0) (HOST array of n_replicas, NULL = zeros) and the MCS clock. */
int32_t kpz_export_packed(kpz_ctx* ctx, void* host_dst, size_t bytes);
int32_t kpz_import_packed(kpz_ctx* ctx, const void* host_src, size_t bytes, const int64_t* h00, uint64_t mcs);

/* End-to-end step with HOST buffers: kpz_import_packed(host_lattice) + kpz_run(mcs) + kpz_measure(...) +
 * kpz_export_packed(host_lattice), i.e. host->device and device->host copies inside the call (bench.py "e2e"). */
int32_t kpz_step_host(kpz_ctx* ctx, void* host_lattice, size_t bytes, int64_t* h00_inout, uint64_t mcs_start,
                      uint64_t mcs, int64_t* sum_h, int64_t* sum_h2, double* W2);

/* kpz_step_host with the copies OVERLAPPED with the kernels for ONE lattice: the
 * lattice travels in n_slabs blocks of rows; as soon as a block has arrived all `mcs` MCS run on the part of it that
 * cannot depend on rows still in flight (dependencies spread by tile + 1 rows per colour pass), rows that are final are
 * copied back while later blocks still compute, and the last stage completes the rest in pass order.  Same kernels,
 * same results as kpz_step_host, bit for bit.  host_lattice should be pinned memory (pageable memory makes the copies
 * synchronous: still correct, no overlap).  The n_slabs blocks ramp up in height (x2) from both ends of the lattice, so that
 * only a short first copy-in and a short last copy-out are exposed; for tile = 64 and 32 they are whole numbers of waves of
 * the tiles the GPU holds at a time (kpz_overlap_plan has the schedule as data).  Needs n_replicas = 1, the default schedule on the tiled
 * kernel, n_slabs >= 2 and every block taller than 8 mcs (tile + 1) + 4 tile rows (n_slabs is reduced until that holds);
 * otherwise it IS kpz_step_host.  Synchronises before returning. */
int32_t kpz_step_host_overlapped(kpz_ctx* ctx, void* host_lattice, size_t bytes, int64_t* h00_inout, uint64_t mcs_start,
                                 uint64_t mcs, uint32_t n_slabs, int64_t* sum_h, int64_t* sum_h2, double* W2);

/* The schedule kpz_step_host_overlapped follows, as plain HOST data (no device, no handle: host logic, checked exhaustively
 * in tests/test_overlap_plan.py).  Inputs: lattice edge L, tile edge (L a multiple of 2 * tile), mcs >= 1 MCS per step,
 * the requested number of blocks n_slabs, wave_tiles = the tiles the GPU holds at a time (SMs x resident tiles per SM; the
 * blocks away from the middle are then whole numbers of such waves, so that their launches end on a full wave; 0: blocks in
 * proportion 1 : 2 : 4 .. : 4 : 2 : 1), and oy[m] < tile, the y offset of the global draw of the m-th MCS of the step
 * (kpz_global_draw).  Outputs, all HOST arrays owned by the caller:
 *   boundaries[*n_stages + 1] : block s holds lattice rows boundaries[s] .. boundaries[s + 1] - 1 (capacity n_slabs + 1)
 *   launches[*n_launches][4]  : in issue order: stage, pass p = 4 m + colour slot, first and last tile row of the
 *                               launch in the shifted frame of MCS m (the last may exceed L / tile - 1: the range wraps);
 *                               the pass runs the tile rows of its colour inside that range (capacity n_slabs * 4 mcs)
 *   copies[*n_copies][3]      : stage, first and last lattice row copied back once that stage has run (capacity n_slabs + 1)
 * *n_stages = 0 (and KPZ_OK) when the shape does not allow the overlap (blocks would be shorter than
 * 8 mcs (tile + 1) + 4 tile rows even for two blocks): kpz_step_host_overlapped then is kpz_step_host.
 * KPZ_EINVAL: NULL pointer, L not a multiple of 2 * tile, mcs = 0, an offset >= tile, n_slabs > 4096. */
int32_t kpz_overlap_plan(uint32_t L, uint32_t tile, uint64_t mcs, uint32_t n_slabs, uint32_t wave_tiles, const uint32_t* oy,
                         int64_t* boundaries, uint32_t* n_stages, int64_t* launches, uint32_t* n_launches, int64_t* copies,
                         uint32_t* n_copies);

/* Pipelined end-to-end steps with HOST buffers: n_lanes independent lattices
 * (same L, p, q, tile, seed as the handle; they differ in state and MCS clock), each a HOST buffer of `bytes` >=
 * lattice_bytes in the device layout above (pinned memory is required for the copies to overlap), are each advanced
 * by `mcs` MCS and measured, n_rounds times over, in the order round 0: lane 0 .. n_lanes-1, round 1: ... .  Each
 * batch is exactly one kpz_step_host (same kernels, same results, bit for bit); what differs is the plumbing: the
 * handle's bound lattice and `device_lattice2` (a second DEVICE buffer of lattice_bytes, 16-byte aligned, owned by
 * the caller) alternate, the host->device copy of batch b+1 and the device->host copy of batch b-1 run on two
 * internal non-blocking streams while the kernels of batch b run on the bound stream.
 *   host_lattices : HOST array of n_lanes HOST pointers; each lattice is overwritten with its advanced state
 *   h00_inout     : HOST [n_lanes][n_replicas] tracked height of site (0,0), in and out (NULL = zeros, not returned)
 *   mcs_start     : HOST [n_lanes] MCS clock of each lane on entry (lane clocks advance by mcs per round)
 *   sum_h, sum_h2, W2 : HOST [n_rounds][n_lanes][n_replicas] out-arrays (any may be NULL), as kpz_measure
 * Synchronises before returning.  Afterwards the handle's own lattice, counters and MCS clock are unspecified:
 * call kpz_init_flat, kpz_set_slopes or kpz_import_packed before using it again.  KPZ_EINVAL for NULL / short /
 * misaligned buffers, n_lanes = 0 or n_rounds = 0; KPZ_EOVERFLOW as kpz_measure (the run completes). */
int32_t kpz_pipeline_host(kpz_ctx* ctx, void* device_lattice2, size_t device_lattice2_bytes, uint32_t n_lanes,
                          void* const* host_lattices, size_t bytes, int64_t* h00_inout, const uint64_t* mcs_start,
                          uint64_t mcs, uint32_t n_rounds, int64_t* sum_h, int64_t* sum_h2, double* W2);

/* ---- power spectrum along the lattice axes (eq. 15-16) ---------------- */

/* Exact integer profiles of replica `replica`: col_sums[x] = sum_y h(x,y), row_sums[y] = sum_x h(x,y) with absolute
 * heights (anchored by h(0,0) like kpz_measure).  HOST out-arrays of length L (either may be NULL).  Synchronises.
 * Any valid L.  These are the only functions of the surface the axis modes of h(k) depend on. */
int32_t kpz_profiles(kpz_ctx* ctx, uint32_t replica, int64_t* col_sums, int64_t* row_sums);

/* Power spectrum S(k) = |h(k)|^2, h(k) = (1/L) sum_x [h(x) - <h>] exp(i k.x) (eq. 15-16 with d = 2), on the two
 * lattice axes, k = 2 pi n / L, n = 0 .. L/2:  Sx[n] = S(k,0), Sy[n] = S(0,k) and their average S[n] ("averaging
 * over x and y directions").  S[0] = 0.  HOST out-arrays of length L/2 + 1 (any may be NULL); one replica,
 * one time: ensemble averages are the caller's sum.  fp64 radix-2 FFT of the two integer profiles on the device.
 * L must be a power of two (KPZ_EINVAL otherwise).  Synchronises.  Does not modify the lattice.
 * Note: the domain decomposition leaves an imprint on S(k) (R18): with the default schedule, narrow peaks
 * at the mode numbers n = (2j+1) L / (2 tile) and n = L/4, a decade above the scaling window 0.002 < k < 0.1 of P:137;
 * kpz_set_sub_sweeps(K >= 2) removes them. */
int32_t kpz_power_spectrum(kpz_ctx* ctx, uint32_t replica, double* S, double* Sx, double* Sy);

/* ---- one lattice split into slabs of rows over several handles / GPUs ------------------
 * For lattices larger than one GPU (L > 2^19), and as the data-parallel form of a single large lattice.  Slab s of
 * n_slabs owns the L / n_slabs lattice rows from row s * L / n_slabs and the tile rows s * NT / n_slabs .. of the
 * shifted frame (NT = L / tile; NT must be a multiple of 2 * n_slabs and L / n_slabs a multiple of 32).  Its buffer
 * stores the owned rows followed by tile + 2 GHOST rows, a copy of the first rows of the next slab (periodically: the
 * last slab's ghost rows are the first rows of slab 0), in the device layout of a whole lattice with L / n_slabs +
 * tile + 2 rows per plane.  The tiles of a slab's last tile row reach oy + 1 rows into the ghost rows (oy = the y
 * origin of the MCS, kpz_global_draw); they are active in the two colour passes whose colour has bit 1 set.  The
 * DRIVER (paper_1110_6745_b200/slabs.py; any code that can copy device memory between the handles) therefore runs,
 * for every MCS m and slot = 0..3 with colour = perm[slot]:
 *     if colour & 2:  copy rows [0, oy + 1) of both planes of slab s+1 into the ghost rows of slab s     (all s)
 *     kpz_slab_pass(slab s, slot)                                                                     (all s)
 *     if colour & 2:  copy the ghost rows [0, oy + 1) of slab s back onto rows [0, oy + 1) of slab s+1  (all s)
 * then kpz_slab_end_mcs on every slab.  The trajectory is the whole-lattice one bit for bit (same tile ids, same
 * streams; tests/test_gpu_parity.py: test_slabs_*).  Default schedule S4 only; one replica.
 * Measurement: kpz_slab_measure_local on every slab (column walks of its owned rows; slab 0 also walks row 0 along
 * x); gather the n_slabs per-column step totals ([n_slabs][L] int32, device) and slab 0's row-0 prefix ([L] int32);
 * kpz_slab_measure_finish on every slab gives four 64-bit half-accumulators; their sums mod 2^64 over the slabs and the
 * sum of the slabs' h(0,0) counters go to kpz_slab_finalize.  kpz_init_flat, kpz_counters (per slab: add them up),
 * kpz_export_packed / kpz_import_packed (the slab's own buffer), kpz_synchronize and kpz_destroy work on slab
 * handles; the calls that address a whole lattice return KPZ_ESTATE. */
int32_t kpz_slab_workspace_bytes(uint32_t L, uint32_t tile, uint32_t n_slabs, size_t* lattice_bytes, size_t* scratch_bytes);
int32_t kpz_create_slab(kpz_ctx** out, uint32_t L, double p, double q, uint32_t tile, uint64_t seed, uint32_t n_slabs,
                        uint32_t slab);
/* HOST out-pointers (any may be NULL): rows owned, rows stored (owned + ghost), bytes of one row of one plane (L / 8),
 * byte offsets INSIDE THE BOUND SCRATCH BUFFER of the row-0 prefix ([L] int32, valid on slab 0 after
 * kpz_slab_measure_local) and of this slab's per-column step totals ([L] int32). */
int32_t kpz_slab_info(const kpz_ctx* ctx, uint32_t* rows_own, uint32_t* rows_stored, size_t* row_bytes, size_t* base_offset,
                      size_t* totals_offset);
/* Global draw S2 of MCS m evaluated on the host (replica 0): origin (ox, oy) and the colour order perm[4] (HOST out). */
int32_t kpz_global_draw(const kpz_ctx* ctx, uint64_t m, uint32_t* ox, uint32_t* oy, uint32_t* perm);
/* Colour pass `slot` (0..3) of the current MCS on this slab's tiles (one launch, asynchronous). */
int32_t kpz_slab_pass(kpz_ctx* ctx, uint32_t slot);
/* Advances this slab's MCS clock by one (after the four passes). */
int32_t kpz_slab_end_mcs(kpz_ctx* ctx);
int32_t kpz_slab_measure_local(kpz_ctx* ctx);
/* d_base0: DEVICE [L] int32 row-0 prefix of slab 0; d_totals_all: DEVICE [n_slabs][L] int32 step totals of all slabs;
 * halves: HOST [4] out.  Synchronises. */
int32_t kpz_slab_measure_finish(kpz_ctx* ctx, const void* d_base0, const void* d_totals_all, uint64_t* halves);
/* halves: HOST [4], summed mod 2^64 over the slabs; h00: sum of the slabs' h(0,0) counters.  Outputs as kpz_measure
 * (HOST, any may be NULL); KPZ_EOVERFLOW as kpz_measure. */
int32_t kpz_slab_finalize(uint32_t L, const uint64_t* halves, int64_t h00, int64_t* sum_h, int64_t* sum_h2, double* W2);

/* Number of kernels this handle has launched since creation (for bench.py "gpu_launches"). */
int32_t kpz_launch_count(const kpz_ctx* ctx, uint64_t* out);

/* Pipe micro-benchmarks for the roofline of the update kernel (MEASURED_PEAKS.json has no
 * integer or shared-memory peak).  Runs, on the CURRENT device, kernels that only issue one kind of instruction from
 * every warp slot of every SM and writes KPZ_N_PEAKS doubles to the HOST array `out` (n >= KPZ_N_PEAKS):
 *   [0] SM clock in Hz during the run (clock64 ticks / globaltimer nanoseconds of one thread)
 *   [1] LOP3, [2] SHF, [3] IMAD, [4] IMAD.WIDE throughput in lane-operations/s (32 per warp instruction)
 *   [5] shared-memory LDS.32 bytes/s with every lane in its own bank (the tile layout of the update kernel)
 *   [6] shared-memory XOR reductions (ATOMS / RED) in lane-operations/s
 *   [7] attempts/s of the bare instruction mix of one p = 1, q = 0 attempt (5 LDS, 2 SHF, 3 LOP3, 1 reduction) issued
 *       without the dependent chain of a real tile -- what the update kernel would reach with perfect latency hiding
 *   [8] number of SMs
 *   [9], [10] SM clocks per attempt and warp of the dependent chain of ONE tile (5 LDS -> 2 SHF -> 3 LOP3 -> XOR
 *       reduction -> the next attempt's loads) with one and with two warps per scheduler on one SM: the latency that
 *       only other resident warps can hide.
 * Takes a few tens of milliseconds.  KPZ_EINVAL for a NULL / short array, KPZ_ECUDA without a device. */
#define KPZ_N_PEAKS 11
int32_t kpz_measure_peaks(double* out, uint32_t n);

/* Tile-layout experiment behind DESIGN.md section 7.1 ("fewer words per tile"): runs, on the CURRENT device, the attempt
 * loop of the T = 64, p = 1, q = 0 kernel ALONE (4096 attempts per tile on tiles of random bits, no staging, nothing
 * written back) in two shared-memory layouts and writes KPZ_N_LAYOUTS doubles to the HOST array `out`:
 *   [0] attempts/s, [1] resident warps per SM: the update kernel's own layout and code (three words per row, 199 words
 *       per tile) -- the ceiling of the present kernel without its staging;
 *   [2] attempts/s, [3] resident warps per SM: tile and halo as one bit string with a row pitch of 66 bits (138 words
 *       per tile): no halo words, but the rows above and below need a rotate each and their own word index.
 * A measurement of a design alternative, not a step of the path.  KPZ_EINVAL for a NULL / short array, KPZ_ECUDA
 * without a device. */
#define KPZ_N_LAYOUTS 4
int32_t kpz_measure_layouts(double* out, uint32_t n);

/* Device Philox4x32-10 self-test: evaluates n (counter,key) inputs on the GPU.  HOST arrays: ctr[4n], key[2n],
 * out[4n].  Used by the tests to check the in-kernel generator against the published known answers. */
int32_t kpz_philox_selftest(const uint32_t* ctr, const uint32_t* key, uint32_t* out, uint32_t n);

#ifdef __cplusplus
}
#endif
#endif /* KPZ_B200_H */
