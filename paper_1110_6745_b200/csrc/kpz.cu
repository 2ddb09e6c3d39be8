// kpz.cu -- host side of libkpz_b200.so: the C ABI of include/kpz.h on top of the kernels in kpz_device.cuh.
// No CPU fallback: every entry point that computes launches CUDA kernels on the bound stream.
#include "kpz_host.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>
#include <vector>

#include "kpz_aux_kernels.cuh"
#include "kpz_peaks.cuh"

namespace {

typedef __int128 i128;
typedef unsigned __int128 u128;

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

ScratchLayout scratch_layout(uint32_t L, uint32_t R) {
    ScratchLayout s;
    // chunks of at most 1024 rows (multiple of 32): chunk-relative sums then fit 32 bits (kpz_column_chunk_kernel)
    uint32_t rpc = L < 1024u ? L : 1024u;
    uint32_t nc = (L + rpc - 1) / rpc;
    s.n_chunks = nc;
    s.rows_per_chunk = rpc;
    size_t o = 0;
    s.stats = o; o += align_up((size_t)R * 4 * 8, 256);
    s.msum = o;  o += align_up((size_t)R * 4 * 8, 256);
    s.misc = o;  o += 256;
    s.base = o;  o += align_up((size_t)R * L * 4, 256);
    s.cS0 = o;   o += align_up((size_t)R * nc * L * 4, 256);
    s.cS1 = o;   o += align_up((size_t)R * nc * L * 4, 256);
    s.cS2 = o;   o += align_up((size_t)R * nc * L * 4, 256);
    s.colsum = o; o += align_up((size_t)L * 8, 256);
    s.rowinc = o; o += align_up((size_t)L * 4, 256);
    s.prof = o;   o += align_up((size_t)2 * L * 8, 256);
    s.fft = o;    o += align_up((size_t)2 * L * 16, 256);
    s.sdir = o;   o += align_up((size_t)2 * (L / 2 + 1) * 8, 256);
    s.savg = o;   o += align_up((size_t)(L / 2 + 1) * 8, 256);
    s.ptab = o;   o += 4096 * 8;
    s.total = o;
    return s;
}

bool valid_tile(uint32_t T) { return T == 4 || T == 8 || T == 16 || T == 32 || T == 64; }

int32_t validate(uint32_t L, double p, double q, uint32_t T, uint32_t R) {
    if (!valid_tile(T)) return KPZ_EINVAL;
    if (L == 0 || L % (2 * T) != 0 || L % 32 != 0) return KPZ_EINVAL;
    if (!(p >= 0.0 && p <= 1.0) || !(q >= 0.0 && q <= 1.0)) return KPZ_EINVAL;
    if (R == 0 || R > 65535u) return KPZ_EINVAL;   // replicas index gridDim.y / gridDim.z of the measurement kernels
    if (L > (1u << 20)) return KPZ_EINVAL;   // int32 heights / tile ids stay in range up to 2^20
    const uint64_t NT = L / T;
    if (NT * NT >= 0xFFFFFFFFull) return KPZ_EINVAL;   // tile_id must never equal the global-draw marker
    return KPZ_OK;
}

uint64_t accept_threshold(double prob) {
    if (prob >= 1.0) return 1ull << 32;
    if (prob <= 0.0) return 0ull;
    return (uint64_t)std::floor(std::ldexp(prob, 32));
}

}  // namespace

namespace {

// Makes the handle's device current for the duration of an entry point and restores the caller's device.
struct DeviceGuard {
    int prev = -1;
    bool changed = false;
    explicit DeviceGuard(int dev) {
        if (dev >= 0 && cudaGetDevice(&prev) == cudaSuccess && prev != dev) changed = (cudaSetDevice(dev) == cudaSuccess);
    }
    ~DeviceGuard() {
        if (changed) cudaSetDevice(prev);
    }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
};

// AUTO takes the resident path up to this many tiles per colour over all replicas (measured cross-over)
constexpr uint64_t KPZ_RESIDENT_AUTO_MAX_TILES = 1u << 20;

int grid_for(uint64_t n, int block, int cap = 148 * 16) {
    uint64_t g = (n + block - 1) / block;
    if (g > (uint64_t)cap) g = cap;
    if (g < 1) g = 1;
    return (int)g;
}

void fill_update_params(const kpz_ctx* c, kpz::UpdateParams& P, uint32_t m, uint32_t slot, uint32_t sub) {
    P.lattice = c->d_lattice;
    P.stats = reinterpret_cast<unsigned long long*>(c->d_scratch + c->sl.stats);
    P.plane_words = (uint64_t)c->L * c->L / 32;
    P.L = c->L;
    P.NT = c->L / c->T;
    P.HN = (c->schedule == KPZ_SCHEDULE_DEAD_BORDER) ? P.NT : P.NT / 2;   // tiles per edge in one launch
    P.W = c->L / 32;
    // whole lattice: all L rows stored, tile rows from 0, rows wrap at L.  A slab handle (kpz_create_slab) stores
    // rows_own + ghost rows from global tile row slab * NT / n_slabs on, never wraps, and runs NT / n_slabs tile rows.
    const bool slab = c->n_slabs > 0;
    P.HNy = slab ? P.NT / c->n_slabs / 2 : P.HN;
    P.ty0 = slab ? c->slab * (P.NT / c->n_slabs) : 0u;
    P.ywrap = slab ? 0xFFFFFFFFu : c->L;
    P.j0 = 0u;
    P.tywrap = slab ? 0xFFFFFFFFu : P.NT;
    if (slab) P.plane_words = (uint64_t)c->rows * (c->L / 32);
    P.tiles_per_colour = P.HN * P.HNy;
    P.total_items = (uint64_t)c->R * P.tiles_per_colour;
    P.blocked = (P.HN % 8 == 0 && P.HNy % 4 == 0) ? 1u : 0u;
    P.thr_p = accept_threshold(c->p);
    P.thr_q = accept_threshold(c->q);
    P.tp_incl = (uint32_t)(P.thr_p - 1);
    P.tq_incl = (uint32_t)(P.thr_q - 1);
    P.m = m;
    P.slot = slot;
    P.sub = sub;
    const uint32_t calls = c->T * c->T / 8u, per = calls / c->sub_sweeps;
    P.call_begin = sub * per;
    P.call_end = (sub + 1u) * per;
    P.pthr = reinterpret_cast<const unsigned long long*>(c->d_scratch + c->sl.ptab);
    P.pn = c->pn;
    P.pk_min = c->pk_min;
    P.key.k0 = (uint32_t)(c->seed & 0xFFFFFFFFull);
    P.key.k1 = (uint32_t)(c->seed >> 32);
}

int32_t launch_update(kpz_ctx* c, uint32_t m, uint32_t slot, uint32_t sub) {
    kpz::UpdateParams P;
    fill_update_params(c, P, m, slot, sub);
    return c->T >= 32 ? kpz_launch_update_wide(c, P) : kpz_launch_update_narrow(c, P);
}

// ---- lattice-resident path (kpz_resident_kernel): one launch for all MCS of a kpz_run call -------------------

size_t tile_words(uint32_t T) {
    switch (T) {
        case 64: return kpz::TileGeom<64>::WORDS;
        case 32: return kpz::TileGeom<32>::WORDS;
        case 16: return kpz::TileGeom<16>::WORDS;
        case 8: return kpz::TileGeom<8>::WORDS;
        default: return kpz::TileGeom<4>::WORDS;
    }
}

ResidentPlan resident_plan(const kpz_ctx* c) {
    ResidentPlan pl{};
    const uint32_t L = c->L, T = c->T;
    const size_t lat = (size_t)L * L / 4;                        // bytes of one packed lattice
    const uint32_t HN = L / T / 2, tpc = HN * HN;
    pl.ok = c->schedule == KPZ_SCHEDULE_COLOURS && !c->poisson && lat <= KPZ_RESIDENT_SMEM_MAX;      // S4, S6
    if (!pl.ok) return pl;
    // threads per CTA: a multiple of 128 wherever the handle has the tiles for it.  Warps are bound to the four
    // schedulers of an SM by their index inside the CTA, so single-warp CTAs would pile every chain of an SM onto
    // one scheduler (measured: 1024 x L = 128 at 32 threads per CTA runs at half the rate of 128 threads per CTA).
    const uint64_t all_tiles = (uint64_t)c->R * tpc;
    pl.nthr = tpc >= 256u ? 256u : (all_tiles >= 128u ? 128u : (all_tiles >= 64u ? 64u : 32u));
    uint32_t G = tpc >= pl.nthr ? 1u : pl.nthr / tpc;
    if (G > c->R) G = c->R;
    const size_t tiles = tile_words(T) * pl.nthr * 4;
    while (G > 1 && G * lat + tiles > KPZ_RESIDENT_SMEM_MAX) --G;
    pl.G = G;
    pl.blocks = (c->R + G - 1) / G;
    pl.smem = G * lat + tiles;
    pl.ok = pl.smem <= KPZ_RESIDENT_SMEM_MAX;
    return pl;
}

int32_t launch_resident(kpz_ctx* c, const ResidentPlan& pl, uint32_t m0, uint32_t n_mcs) {
    kpz::UpdateParams P;
    fill_update_params(c, P, m0, 0u, 0u);
    return c->T >= 32 ? kpz_launch_resident_wide(c, P, pl, n_mcs) : kpz_launch_resident_narrow(c, P, pl, n_mcs);
}

// Which kernels advance the lattice.  AUTO: the resident kernel when the packed lattice fits in shared memory
// (L <= 512 in practice) and a colour has too few tiles to fill the GPU, else the tiled kernel.
int32_t choose_path(kpz_ctx* c, ResidentPlan& pl) {
    if (c->path == KPZ_PATH_TILED) return KPZ_PATH_TILED;
    pl = resident_plan(c);
    if (c->path == KPZ_PATH_RESIDENT) return pl.ok ? KPZ_PATH_RESIDENT : -1;
    if (!pl.ok) return KPZ_PATH_TILED;
    const uint64_t tpc = (uint64_t)(c->L / c->T / 2) * (c->L / c->T / 2);
    return ((uint64_t)c->R * tpc <= KPZ_RESIDENT_AUTO_MAX_TILES) ? KPZ_PATH_RESIDENT : KPZ_PATH_TILED;
}

int32_t require_bound(kpz_ctx* c) {
    if (!c) return KPZ_EINVAL;
    if (!c->bound) return kpz_fail(c, KPZ_ESTATE, "kpz_bind has not been called");
    return KPZ_OK;
}

// entry points that address the lattice as a whole (windows, hash, profiles, kpz_run, kpz_measure ...)
int32_t require_whole(kpz_ctx* c) {
    if (c->n_slabs > 0) return kpz_fail(c, KPZ_ESTATE, "not available on a slab handle (use the kpz_slab_* calls)");
    return KPZ_OK;
}

// host evaluation of the global draw S2 (the kernels evaluate the same draw in-kernel; the slab driver needs the
// origin and the colour order to know which rows to exchange)
void host_philox4x32_10(uint32_t c[4], uint32_t k0, uint32_t k1) {
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c[0], p1 = (uint64_t)0xCD9E8D57u * c[2];
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c[1] ^ k0, n2 = (uint32_t)(p0 >> 32) ^ c[3] ^ k1;
        c[1] = (uint32_t)p1; c[3] = (uint32_t)p0; c[0] = n0; c[2] = n2;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
}

void host_global_draw(const kpz_ctx* c, uint32_t m, uint32_t sub, uint32_t replica, uint32_t* ox, uint32_t* oy, uint32_t perm[4]) {
    uint32_t G[4] = {sub, 0xFFFFFFFFu, m, replica};
    host_philox4x32_10(G, (uint32_t)(c->seed & 0xFFFFFFFFull), (uint32_t)(c->seed >> 32));
    const uint32_t g = 4, T = c->T;
    *ox = g * (uint32_t)(((uint64_t)G[0] * (T / g)) >> 32);
    *oy = g * (uint32_t)(((uint64_t)G[1] * (T / g)) >> 32);
    const uint32_t pidx = (uint32_t)(((uint64_t)G[2] * 24u) >> 32);
    const uint32_t d[3] = {pidx / 6u, (pidx % 6u) / 2u, pidx % 2u};
    uint32_t pool[4] = {0, 1, 2, 3};
    int n = 4;
    for (int k = 0; k < 3; ++k) {
        perm[k] = pool[d[k]];
        for (int j = (int)d[k]; j < n - 1; ++j) pool[j] = pool[j + 1];
        --n;
    }
    perm[3] = pool[0];
}

// sum h, sum h^2, W^2 of one lattice from the sums relative to h(0,0) (R16: 128-bit integers, one conversion, one division)
bool finalize_sums(uint32_t L, i128 S1, i128 S2, long long h00, int64_t* sum_h, int64_t* sum_h2, double* W2);

// sums for all replicas -> host vectors (relative to h(0,0)) + h00
int32_t measure_relative(kpz_ctx* c, std::vector<i128>& S1, std::vector<i128>& S2, std::vector<long long>& h00,
                         bool want_colsum = false, uint32_t colsum_replica = 0) {
    const uint32_t L = c->L, R = c->R, W = L / 32;
    const uint64_t plane_words = (uint64_t)L * L / 32;
    unsigned char* sc = c->d_scratch;
    unsigned long long* msum = reinterpret_cast<unsigned long long*>(sc + c->sl.msum);
    int32_t* base = reinterpret_cast<int32_t*>(sc + c->sl.base);
    int32_t* cS0 = reinterpret_cast<int32_t*>(sc + c->sl.cS0);
    int32_t* cS1 = reinterpret_cast<int32_t*>(sc + c->sl.cS1);
    int32_t* cS2 = reinterpret_cast<int32_t*>(sc + c->sl.cS2);
    KPZ_CUDA(c, cudaMemsetAsync(msum, 0, (size_t)R * 32, c->stream));
    int nthr = 1024;
    while (nthr > 32 && (uint32_t)nthr > L) nthr >>= 1;
    kpz::kpz_row0_prefix_kernel<<<R, nthr, 0, c->stream>>>(c->d_lattice, plane_words, L, W, base);
    KPZ_CUDA(c, cudaGetLastError());
    dim3 g1((W + 127) / 128, c->sl.n_chunks, R);
    kpz::kpz_column_chunk_kernel<<<g1, 128, 0, c->stream>>>(c->d_lattice, plane_words, L, W, c->sl.rows_per_chunk, cS0,
                                                         cS1, cS2, L, 1u);
    KPZ_CUDA(c, cudaGetLastError());
    dim3 g2((L + 255) / 256, R);
    kpz::kpz_combine_kernel<<<g2, 256, 0, c->stream>>>(base, cS0, cS1, cS2, L, c->sl.n_chunks, c->sl.rows_per_chunk, msum,
                                                    want_colsum ? reinterpret_cast<long long*>(sc + c->sl.colsum) : nullptr,
                                                    colsum_replica, L);
    KPZ_CUDA(c, cudaGetLastError());
    c->launches += 3;
    std::vector<unsigned long long> hm((size_t)R * 4), hs((size_t)R * 4);
    KPZ_CUDA(c, cudaMemcpyAsync(hm.data(), msum, (size_t)R * 32, cudaMemcpyDeviceToHost, c->stream));
    KPZ_CUDA(c, cudaMemcpyAsync(hs.data(), sc + c->sl.stats, (size_t)R * 32, cudaMemcpyDeviceToHost, c->stream));
    KPZ_CUDA(c, cudaStreamSynchronize(c->stream));
    S1.resize(R); S2.resize(R); h00.resize(R);
    for (uint32_t r = 0; r < R; ++r) {
        S1[r] = (i128)(long long)hm[4 * r + 1] * ((i128)1 << 32) + (i128)hm[4 * r + 0];
        S2[r] = (i128)(long long)hm[4 * r + 3] * ((i128)1 << 32) + (i128)hm[4 * r + 2];
        h00[r] = (long long)hs[4 * r + 2];
    }
    return KPZ_OK;
}

bool fits_i64(i128 v) { return v >= (i128)INT64_MIN && v <= (i128)INT64_MAX; }

// returns true if a requested int64 output overflowed (it is then written as 0)
bool finalize_sums(uint32_t L, i128 S1, i128 S2, long long h00, int64_t* sum_h, int64_t* sum_h2, double* W2) {
    const i128 N = (i128)L * L;
    const double Nd = (double)((uint64_t)L * L);
    const i128 h0 = h00;
    const i128 sh = S1 + N * h0;                          // sum h
    const i128 sh2 = S2 + 2 * h0 * S1 + N * h0 * h0;      // sum h^2
    // N*sum_h2 - sum_h^2 is invariant under the shift by h0: evaluate it on the small relative sums
    const i128 num = N * S2 - S1 * S1;
    bool overflow = false;
    if (W2) *W2 = (double)num / (Nd * Nd);
    if (sum_h) { if (fits_i64(sh)) *sum_h = (int64_t)sh; else { *sum_h = 0; overflow = true; } }
    if (sum_h2) { if (fits_i64(sh2)) *sum_h2 = (int64_t)sh2; else { *sum_h2 = 0; overflow = true; } }
    return overflow;
}

}  // namespace

namespace {

template <int KIND>
cudaError_t run_peak(uint32_t blocks, uint32_t iters, uint32_t* sink, unsigned long long* ticks, float* ms) {
    cudaEvent_t e0, e1;
    cudaError_t e = cudaEventCreate(&e0);
    if (e != cudaSuccess) return e;
    e = cudaEventCreate(&e1);
    if (e != cudaSuccess) { cudaEventDestroy(e0); return e; }
    kpz::kpz_peak_kernel<KIND><<<blocks, 256>>>(iters / 8 + 1, 0x9E3779B9u, sink, ticks);      // warm-up
    float best = 1e30f;
    for (int rep = 0; rep < 3 && e == cudaSuccess; ++rep) {
        cudaEventRecord(e0);
        kpz::kpz_peak_kernel<KIND><<<blocks, 256>>>(iters, 0x9E3779B9u + rep, sink, ticks);
        cudaEventRecord(e1);
        e = cudaEventSynchronize(e1);
        float t = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&t, e0, e1);
        if (e == cudaSuccess && t < best) best = t;
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *ms = best;
    return e;
}

// the attempt loop of T = 64 alone in tile layout LAYOUT (kpz_peaks.cuh): attempts/s with `waves` CTAs per CTA slot
template <int LAYOUT>
cudaError_t run_layout(int sms, uint32_t* sink, double* attempts_per_s, double* warps_per_sm) {
    constexpr int NTHR = 96;
    const size_t smem = (size_t)(LAYOUT ? kpz::LAYOUT66_WORDS : kpz::TileGeom<64>::WORDS) * NTHR * sizeof(uint32_t);
    cudaError_t e = cudaFuncSetAttribute(kpz::kpz_layout_kernel<LAYOUT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kpz::kpz_layout_kernel<LAYOUT>, NTHR, smem);
    if (e != cudaSuccess) return e;
    if (per_sm <= 0) return cudaErrorInvalidConfiguration;
    *warps_per_sm = per_sm * (NTHR / 32.0);
    const uint32_t blocks = (uint32_t)(sms * per_sm * 8);        // eight full waves
    cudaEvent_t e0, e1;
    e = cudaEventCreate(&e0);
    if (e != cudaSuccess) return e;
    e = cudaEventCreate(&e1);
    if (e != cudaSuccess) { cudaEventDestroy(e0); return e; }
    kpz::kpz_layout_kernel<LAYOUT><<<blocks, NTHR, smem>>>(0x9E3779B9u, 1u, 2u, 1u << 27, sink);      // warm-up
    float best = 1e30f;
    for (int rep = 0; rep < 3 && e == cudaSuccess; ++rep) {
        cudaEventRecord(e0);
        kpz::kpz_layout_kernel<LAYOUT><<<blocks, NTHR, smem>>>(0x9E3779B9u + rep, 2u + rep, 2u, 1u << 27, sink);
        cudaEventRecord(e1);
        e = cudaEventSynchronize(e1);
        float t = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&t, e0, e1);
        if (e == cudaSuccess && t < best) best = t;
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    *attempts_per_s = (double)blocks * NTHR * 4096.0 / (best * 1e-3);
    return e;
}

// ---- kpz_measure_static: the measurement with its scratch in a file-scope static array (no allocation) ----------
// For callers that cannot allocate (code under CUDA graph capture, tight serving loops).  The partial sums of the
// measurement kernels -- row-0 prefix, per-chunk (S0, S1, S2) of every column, the four 64-bit half-accumulators --
// live in this array instead of the caller's scratch buffer.  Every GPU that loads the library holds it until exit.
// Maximum lattice edge KPZ_STATIC_MAX_L = 8192 (include/kpz.h; the paper's largest steady-state size): 819 456 bytes.
// Layout (bytes): [0, 256) four u64 half-accumulators; base[L_max] int32; cS0, cS1, cS2 [NC_max][L_max] int32 each.
constexpr uint32_t KPZ_STATIC_MAX_CHUNKS = KPZ_STATIC_MAX_L / 1024;      // KPZ_STATIC_MAX_L: include/kpz.h
constexpr size_t KPZ_STATIC_OFF_BASE = 256;
constexpr size_t KPZ_STATIC_OFF_CS = KPZ_STATIC_OFF_BASE + (size_t)KPZ_STATIC_MAX_L * 4;
constexpr size_t KPZ_STATIC_CS_BYTES = (size_t)KPZ_STATIC_MAX_CHUNKS * KPZ_STATIC_MAX_L * 4;
constexpr size_t KPZ_STATIC_BYTES = KPZ_STATIC_OFF_CS + 3 * KPZ_STATIC_CS_BYTES;
static __device__ __align__(256) unsigned char kpz_static_scratch[KPZ_STATIC_BYTES];

// Device code may name the array directly.  One thread: half-accumulators -> sum h, sum h^2, W^2 (same 128-bit integer
// arithmetic as the host's finalize_sums: R16) written to the caller's DEVICE buffer out[8]:
//   [0..3] the half-accumulators (lo / hi of sum (h - h00), lo / hi of sum (h - h00)^2)
//   [4] sum h (int64), [5] sum h^2 (int64), [6] W^2 (double), [7] 1 if a sum does not fit int64 (it is then 0) else 0
__global__ void kpz_static_finalize_kernel(const unsigned long long* __restrict__ stats, uint32_t replica, uint32_t L,
                                           unsigned long long* __restrict__ out) {
    if (blockIdx.x != 0 || threadIdx.x != 0) return;
    const unsigned long long* hm = reinterpret_cast<const unsigned long long*>(kpz_static_scratch);
    const i128 S1 = (i128)(long long)hm[1] * ((i128)1 << 32) + (i128)hm[0];
    const i128 S2 = (i128)(long long)hm[3] * ((i128)1 << 32) + (i128)hm[2];
    const i128 h0 = (long long)stats[(size_t)replica * 4u + 2u];
    const i128 N = (i128)L * L;
    const double Nd = (double)((unsigned long long)L * L);
    const i128 sh = S1 + N * h0;
    const i128 sh2 = S2 + 2 * h0 * S1 + N * h0 * h0;
    const i128 num = N * S2 - S1 * S1;
    const i128 lo = -((i128)1 << 63), hi = ((i128)1 << 63) - 1;
    const bool ok1 = sh >= lo && sh <= hi, ok2 = sh2 >= lo && sh2 <= hi;
    out[0] = hm[0]; out[1] = hm[1]; out[2] = hm[2]; out[3] = hm[3];
    out[4] = ok1 ? (unsigned long long)(long long)sh : 0ull;
    out[5] = ok2 ? (unsigned long long)(long long)sh2 : 0ull;
    out[6] = (unsigned long long)__double_as_longlong((double)num / (Nd * Nd));
    out[7] = (ok1 && ok2) ? 0ull : 1ull;
}

// In host code the array's name is a host-side stand-in, not a device address: look the address up once per device,
// with that device current, and hand THAT to the kernels.
int32_t static_scratch_ptr(kpz_ctx* c, unsigned char** out) {
    static unsigned char* ptr[KPZ_MAX_DEVICES] = {};
    const int dev = c->device;
    if (dev < 0 || dev >= KPZ_MAX_DEVICES) return kpz_fail(c, KPZ_ESTATE, "handle has no device");
    if (!ptr[dev]) {
        unsigned char* p = nullptr;
        KPZ_CUDA(c, cudaGetSymbolAddress((void**)&p, kpz_static_scratch));      // the caller made `dev` current
        if (!p) return kpz_fail(c, KPZ_ECUDA, "cudaGetSymbolAddress returned a NULL address");
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return KPZ_OK;
}

}  // namespace

extern "C" {

int32_t kpz_workspace_bytes(uint32_t L, uint32_t tile, uint32_t n_replicas, size_t* lattice_bytes,
                            size_t* scratch_bytes) {
    int32_t rc = validate(L, 0.0, 0.0, tile, n_replicas);
    if (rc != KPZ_OK) return rc;
    if (lattice_bytes) *lattice_bytes = (size_t)n_replicas * ((size_t)L * L / 4);
    if (scratch_bytes) *scratch_bytes = scratch_layout(L, n_replicas).total;
    return KPZ_OK;
}

int32_t kpz_create_batch(kpz_ctx** out, uint32_t L, double p, double q, uint32_t tile, uint64_t seed,
                         uint32_t n_replicas) {
    if (!out) return KPZ_EINVAL;
    *out = nullptr;
    int32_t rc = validate(L, p, q, tile, n_replicas);
    if (rc != KPZ_OK) return rc;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0) return KPZ_ECUDA;   // no CPU fallback
    kpz_ctx* c = new (std::nothrow) kpz_ctx();
    if (!c) return KPZ_ENOMEM;
    c->L = L; c->T = tile; c->R = n_replicas; c->p = p; c->q = q; c->seed = seed;
    c->mcs = 0; c->launches = 0; c->schedule = KPZ_SCHEDULE_COLOURS; c->sub_sweeps = 1;
    c->poisson = false; c->pn = 0; c->pk_min = 0; c->attempts_base = 0; c->path = KPZ_PATH_AUTO;
    c->d_lattice = nullptr; c->d_scratch = nullptr; c->stream = nullptr; c->bound = false; c->device = -1; c->s_in = nullptr; c->s_out = nullptr;
    c->n_slabs = 0; c->slab = 0; c->rows_own = L; c->rows = L;
    c->sl = scratch_layout(L, n_replicas);
    c->lattice_bytes = (size_t)n_replicas * ((size_t)L * L / 4);
    c->err[0] = 0;
    *out = c;
    return KPZ_OK;
}

int32_t kpz_create(kpz_ctx** out, uint32_t L, double p, double q, uint32_t tile, uint64_t seed) {
    return kpz_create_batch(out, L, p, q, tile, seed, 1);
}

int32_t kpz_bind(kpz_ctx* c, void* d_lattice, size_t lattice_bytes, void* d_scratch, size_t scratch_bytes,
                 void* cuda_stream) {
    if (!c) return KPZ_EINVAL;
    if (!d_lattice || !d_scratch) return kpz_fail(c, KPZ_EINVAL, "NULL device buffer");
    if (lattice_bytes < c->lattice_bytes || scratch_bytes < c->sl.total)
        return kpz_fail(c, KPZ_ENOMEM, "bound buffers too small: need %zu + %zu bytes", c->lattice_bytes, c->sl.total);
    if (((uintptr_t)d_lattice & 15u) || ((uintptr_t)d_scratch & 15u)) return kpz_fail(c, KPZ_EINVAL, "buffers must be 16-byte aligned");
    // the device is the one that owns the buffers, whatever device is current in the calling thread
    cudaPointerAttributes al, as;
    KPZ_CUDA(c, cudaPointerGetAttributes(&al, d_lattice));
    KPZ_CUDA(c, cudaPointerGetAttributes(&as, d_scratch));
    if (al.type != cudaMemoryTypeDevice || as.type != cudaMemoryTypeDevice || al.device != as.device)
        return kpz_fail(c, KPZ_EINVAL, "lattice and scratch must be device memory of one device");
    if (al.device < 0 || al.device >= KPZ_MAX_DEVICES) return kpz_fail(c, KPZ_EINVAL, "device ordinal out of range");
    c->device = al.device;
    DeviceGuard dg__(c->device);
    c->d_lattice = static_cast<uint32_t*>(d_lattice);
    c->d_scratch = static_cast<unsigned char*>(d_scratch);
    c->stream = static_cast<cudaStream_t>(cuda_stream);
    KPZ_CUDA(c, cudaMemsetAsync(c->d_scratch, 0, c->sl.base, c->stream));   // counters, sums, misc
    c->bound = true;
    return KPZ_OK;
}

int32_t kpz_init_flat(kpz_ctx* c) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    const uint64_t n_words = c->lattice_bytes / 4;      // both planes of every replica (of the stored rows of a slab)
    kpz::kpz_fill_flat_kernel<<<grid_for(n_words, 256, 148 * 32), 256, 0, c->stream>>>(c->d_lattice, n_words, c->L / 32);
    KPZ_CUDA(c, cudaGetLastError());
    c->launches++;
    KPZ_CUDA(c, cudaMemsetAsync(c->d_scratch + c->sl.stats, 0, (size_t)c->R * 32, c->stream));
    c->mcs = 0;
    c->attempts_base = 0;
    return KPZ_OK;
}

int32_t kpz_run(kpz_ctx* c, uint64_t mcs) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if ((rc = require_whole(c)) != KPZ_OK) return rc;
    if (c->mcs + mcs > 0xFFFFFFFFull) return kpz_fail(c, KPZ_EINVAL, "MCS clock would exceed 2^32-1");
    if (mcs == 0) return KPZ_OK;
    ResidentPlan pl{};
    const int32_t path = choose_path(c, pl);
    if (path < 0) return kpz_fail(c, KPZ_EINVAL, "the resident path needs a lattice that fits in shared memory and the default schedule");
    if (path != KPZ_PATH_TILED) {
        rc = launch_resident(c, pl, (uint32_t)c->mcs, (uint32_t)mcs);
        if (rc != KPZ_OK) return rc;
        c->mcs += mcs;
        c->attempts_base += mcs * (uint64_t)c->L * c->L;
        return KPZ_OK;
    }
    for (uint64_t k = 0; k < mcs; ++k) {
        const uint32_t m = (uint32_t)c->mcs;
        const uint32_t passes = (c->schedule == KPZ_SCHEDULE_DEAD_BORDER) ? 1u : 4u;
        for (uint32_t sub = 0; sub < c->sub_sweeps; ++sub) {
            for (uint32_t slot = 0; slot < passes; ++slot) {
                rc = launch_update(c, m, slot, sub);
                if (rc != KPZ_OK) return rc;
            }
        }
        c->mcs++;
        if (!c->poisson) c->attempts_base += (uint64_t)c->L * c->L;
    }
    return KPZ_OK;
}

int32_t kpz_set_path(kpz_ctx* c, int32_t path) {
    if (!c) return KPZ_EINVAL;
    if (path < KPZ_PATH_AUTO || path > KPZ_PATH_RESIDENT) return kpz_fail(c, KPZ_EINVAL, "unknown path");
    c->path = path;
    return KPZ_OK;
}

int32_t kpz_set_schedule(kpz_ctx* c, int32_t schedule) {
    if (!c) return KPZ_EINVAL;
    if (schedule != KPZ_SCHEDULE_COLOURS && schedule != KPZ_SCHEDULE_DEAD_BORDER) return kpz_fail(c, KPZ_EINVAL, "unknown schedule");
    c->schedule = schedule;
    return KPZ_OK;
}

static int32_t upload_poisson_table(kpz_ctx* c);

int32_t kpz_set_sub_sweeps(kpz_ctx* c, uint32_t K) {
    if (!c) return KPZ_EINVAL;
    const uint32_t calls = c->T * c->T / 8u;
    if (K < 1 || K > calls || calls % K != 0) return kpz_fail(c, KPZ_EINVAL, "sub-sweeps must divide tile*tile/8");
    c->sub_sweeps = K;
    DeviceGuard dg__(c->device);
    return (c->poisson && c->bound) ? upload_poisson_table(c) : KPZ_OK;
}

// S7 table: weights 2^52 at the mode, floor-multiplied down both sides, thresholds in 2^-32
static int32_t upload_poisson_table(kpz_ctx* c) {
    const uint64_t lam = (uint64_t)c->T * c->T / c->sub_sweeps;
    uint64_t W = 0;
    while (W * W < 144ull * lam) ++W;
    W += 16;
    const uint64_t kmin = lam > W ? lam - W : 0, kmax = lam + W, n = kmax - kmin + 1;
    if (n > 4096) return kpz_fail(c, KPZ_EINVAL, "Poisson table too large");
    std::vector<u128> w(n);
    w[lam - kmin] = (u128)1 << 52;
    for (uint64_t k = lam + 1; k <= kmax; ++k) w[k - kmin] = w[k - kmin - 1] * lam / k;
    for (uint64_t k = lam; k > kmin; --k) w[k - 1 - kmin] = w[k - kmin] * k / lam;
    u128 total = 0;
    for (uint64_t i = 0; i < n; ++i) total += w[i];
    std::vector<unsigned long long> thr(n);
    u128 run = 0;
    for (uint64_t i = 0; i < n; ++i) {
        run += w[i];
        thr[i] = (unsigned long long)((run << 32) / total);
    }
    KPZ_CUDA(c, cudaMemcpyAsync(c->d_scratch + c->sl.ptab, thr.data(), n * 8, cudaMemcpyHostToDevice, c->stream));
    KPZ_CUDA(c, cudaStreamSynchronize(c->stream));
    c->pn = (uint32_t)n;
    c->pk_min = (uint32_t)kmin;
    return KPZ_OK;
}

int32_t kpz_set_poisson(kpz_ctx* c, int32_t on) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if ((rc = require_whole(c)) != KPZ_OK) return rc;
    c->poisson = on != 0;
    return c->poisson ? upload_poisson_table(c) : KPZ_OK;
}

int32_t kpz_measure(kpz_ctx* c, int64_t* sum_h, int64_t* sum_h2, double* W2) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if ((rc = require_whole(c)) != KPZ_OK) return rc;
    std::vector<i128> S1, S2;
    std::vector<long long> h00;
    rc = measure_relative(c, S1, S2, h00);
    if (rc != KPZ_OK) return rc;
    bool overflow = false;
    for (uint32_t r = 0; r < c->R; ++r)
        overflow |= finalize_sums(c->L, S1[r], S2[r], h00[r], sum_h ? sum_h + r : nullptr, sum_h2 ? sum_h2 + r : nullptr,
                                  W2 ? W2 + r : nullptr);
    if (overflow) return kpz_fail(c, KPZ_EOVERFLOW, "a sum does not fit int64");
    return KPZ_OK;
}

int32_t kpz_measure_static(kpz_ctx* c, uint32_t replica, void* d_out) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if ((rc = require_whole(c)) != KPZ_OK) return rc;
    if (replica >= c->R) return kpz_fail(c, KPZ_EINVAL, "replica out of range");
    if (!d_out || ((uintptr_t)d_out & 7u)) return kpz_fail(c, KPZ_EINVAL, "d_out must be an 8-byte aligned DEVICE pointer to 64 bytes");
    if (c->L > KPZ_STATIC_MAX_L)
        return kpz_fail(c, KPZ_EINVAL, "kpz_measure_static: L = %u exceeds the static scratch maximum of L = %u (use kpz_measure)",
                        c->L, (uint32_t)KPZ_STATIC_MAX_L);
    unsigned char* sp = nullptr;
    if ((rc = static_scratch_ptr(c, &sp)) != KPZ_OK) return rc;
    const uint32_t L = c->L, W = L / 32;
    const uint64_t plane_words = (uint64_t)L * L / 32;
    const uint32_t* lat = c->d_lattice + (size_t)replica * 2u * plane_words;      // this replica's two planes
    unsigned long long* msum = reinterpret_cast<unsigned long long*>(sp);
    int32_t* base = reinterpret_cast<int32_t*>(sp + KPZ_STATIC_OFF_BASE);
    int32_t* cS0 = reinterpret_cast<int32_t*>(sp + KPZ_STATIC_OFF_CS);
    int32_t* cS1 = reinterpret_cast<int32_t*>(sp + KPZ_STATIC_OFF_CS + KPZ_STATIC_CS_BYTES);
    int32_t* cS2 = reinterpret_cast<int32_t*>(sp + KPZ_STATIC_OFF_CS + 2 * KPZ_STATIC_CS_BYTES);
    // the array keeps the last call's contents: the accumulators must start at zero (base and the chunk partials are
    // overwritten in full for this L before they are read)
    KPZ_CUDA(c, cudaMemsetAsync(msum, 0, 32, c->stream));
    int nthr = 1024;
    while (nthr > 32 && (uint32_t)nthr > L) nthr >>= 1;
    kpz::kpz_row0_prefix_kernel<<<1, nthr, 0, c->stream>>>(lat, plane_words, L, W, base);
    KPZ_CUDA(c, cudaGetLastError());
    dim3 g1((W + 127) / 128, c->sl.n_chunks, 1);
    kpz::kpz_column_chunk_kernel<<<g1, 128, 0, c->stream>>>(lat, plane_words, L, W, c->sl.rows_per_chunk, cS0, cS1, cS2, L, 1u);
    KPZ_CUDA(c, cudaGetLastError());
    dim3 g2((L + 255) / 256, 1);
    kpz::kpz_combine_kernel<<<g2, 256, 0, c->stream>>>(base, cS0, cS1, cS2, L, c->sl.n_chunks, c->sl.rows_per_chunk, msum, nullptr,
                                                    0u, L);
    KPZ_CUDA(c, cudaGetLastError());
    kpz_static_finalize_kernel<<<1, 32, 0, c->stream>>>(reinterpret_cast<const unsigned long long*>(c->d_scratch + c->sl.stats), replica,
                                                     L, static_cast<unsigned long long*>(d_out));
    KPZ_CUDA(c, cudaGetLastError());
    c->launches += 4;
    return KPZ_OK;
}

int32_t kpz_run_sampled(kpz_ctx* c, const uint64_t* times, uint32_t n_times, int64_t* sum_h, int64_t* sum_h2, double* W2) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if (!times || n_times == 0) return kpz_fail(c, KPZ_EINVAL, "no sampling times");
    uint64_t prev = c->mcs;
    for (uint32_t i = 0; i < n_times; ++i) {
        if (times[i] < prev || (i > 0 && times[i] == times[i - 1])) return kpz_fail(c, KPZ_EINVAL, "sampling times must increase from the current MCS clock");
        prev = times[i];
    }
    int32_t worst = KPZ_OK;
    for (uint32_t i = 0; i < n_times; ++i) {
        rc = kpz_run(c, times[i] - c->mcs);
        if (rc != KPZ_OK) return rc;
        const size_t o = (size_t)i * c->R;
        rc = kpz_measure(c, sum_h ? sum_h + o : nullptr, sum_h2 ? sum_h2 + o : nullptr, W2 ? W2 + o : nullptr);
        if (rc == KPZ_EOVERFLOW) worst = rc;
        else if (rc != KPZ_OK) return rc;
    }
    return worst;
}

int32_t kpz_destroy(kpz_ctx* c) {
    if (c) {
        DeviceGuard dg__(c->device);
        for (cudaEvent_t e : c->events) cudaEventDestroy(e);
        if (c->s_in) cudaStreamDestroy(c->s_in);
        if (c->s_out) cudaStreamDestroy(c->s_out);
    }
    delete c;
    return KPZ_OK;
}

int32_t kpz_synchronize(kpz_ctx* c) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    KPZ_CUDA(c, cudaStreamSynchronize(c->stream));
    return KPZ_OK;
}

const char* kpz_last_error(const kpz_ctx* c) { return c ? c->err : "null handle"; }

int32_t kpz_get_window(kpz_ctx* c, uint32_t replica, uint32_t x0, uint32_t y0, uint32_t w, uint32_t h, int8_t* sx,
                       int8_t* sy) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if ((rc = require_whole(c)) != KPZ_OK) return rc;
    if (replica >= c->R || !sx || !sy || w == 0 || h == 0 || w > c->L || h > c->L) return kpz_fail(c, KPZ_EINVAL, "bad window");
    const size_t n = (size_t)w * h;
    int8_t* d = nullptr;
    if (cudaMalloc(&d, 2 * n) != cudaSuccess) { cudaGetLastError(); return kpz_fail(c, KPZ_ENOMEM, "temporary device buffer"); }
    kpz::kpz_unpack_window_kernel<<<grid_for(n, 256), 256, 0, c->stream>>>(c->d_lattice, (uint64_t)c->L * c->L / 32, replica,
                                                                       c->L, c->L / 32, x0 % c->L, y0 % c->L, w, h, d, d + n);
    cudaError_t e = cudaGetLastError();
    c->launches++;
    if (e == cudaSuccess) e = cudaMemcpyAsync(sx, d, n, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(sy, d + n, n, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    cudaFree(d);
    if (e != cudaSuccess) return kpz_fail(c, KPZ_ECUDA, "get_window: %s", cudaGetErrorString(e));
    return KPZ_OK;
}

int32_t kpz_get_slopes(kpz_ctx* c, uint32_t replica, int8_t* sx, int8_t* sy) {
    if (!c) return KPZ_EINVAL;
    return kpz_get_window(c, replica, 0, 0, c->L, c->L, sx, sy);
}

int32_t kpz_set_slopes(kpz_ctx* c, uint32_t replica, const int8_t* sx, const int8_t* sy, int64_t h00) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if ((rc = require_whole(c)) != KPZ_OK) return rc;
    if (replica >= c->R || !sx || !sy) return kpz_fail(c, KPZ_EINVAL, "bad argument");
    const size_t n = (size_t)c->L * c->L;
    int8_t* d = nullptr;
    if (cudaMalloc(&d, 2 * n) != cudaSuccess) { cudaGetLastError(); return kpz_fail(c, KPZ_ENOMEM, "temporary device buffer"); }
    int* flags = reinterpret_cast<int*>(c->d_scratch + c->sl.misc + 8);
    int hflags = 0;
    cudaError_t e = cudaMemcpyAsync(d, sx, n, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d + n, sy, n, cudaMemcpyHostToDevice, c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(flags, 0, sizeof(int), c->stream);
    if (e == cudaSuccess) {
        kpz::kpz_validate_kernel<<<grid_for(n, 256), 256, 0, c->stream>>>(d, d + n, c->L, flags);
        c->launches++;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(&hflags, flags, sizeof(int), cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e == cudaSuccess && hflags == 0) {
        kpz::kpz_pack_kernel<<<grid_for(n / 32, 256), 256, 0, c->stream>>>(c->d_lattice, (uint64_t)n / 32, replica, c->L,
                                                                      c->L / 32, d, d + n);
        c->launches++;
        e = cudaGetLastError();
        long long hv = h00;
        if (e == cudaSuccess)
            e = cudaMemcpyAsync(c->d_scratch + c->sl.stats + (size_t)replica * 32 + 16, &hv, 8, cudaMemcpyHostToDevice, c->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    }
    cudaFree(d);
    if (e != cudaSuccess) return kpz_fail(c, KPZ_ECUDA, "set_slopes: %s", cudaGetErrorString(e));
    if (hflags & 1) return kpz_fail(c, KPZ_EINVAL, "slopes must be +1 or -1");
    if (hflags) return kpz_fail(c, KPZ_ESTATE, "state is not curl-free with zero tilt (flags %d)", hflags);
    return KPZ_OK;
}

int32_t kpz_state_hash(kpz_ctx* c, uint32_t replica, uint64_t* out) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if ((rc = require_whole(c)) != KPZ_OK) return rc;
    if (replica >= c->R || !out) return kpz_fail(c, KPZ_EINVAL, "bad argument");
    unsigned long long* acc = reinterpret_cast<unsigned long long*>(c->d_scratch + c->sl.misc);
    const uint64_t plane_words = (uint64_t)c->L * c->L / 32;
    KPZ_CUDA(c, cudaMemsetAsync(acc, 0, 8, c->stream));
    kpz::kpz_hash_kernel<<<grid_for(plane_words, 256), 256, 0, c->stream>>>(c->d_lattice, plane_words, replica, c->L, c->L / 32, acc);
    KPZ_CUDA(c, cudaGetLastError());
    c->launches++;
    unsigned long long h = 0;
    KPZ_CUDA(c, cudaMemcpyAsync(&h, acc, 8, cudaMemcpyDeviceToHost, c->stream));
    KPZ_CUDA(c, cudaStreamSynchronize(c->stream));
    *out = h;
    return KPZ_OK;
}

int32_t kpz_counters(kpz_ctx* c, uint32_t replica, uint64_t* attempts, uint64_t* deposits, uint64_t* removals,
                     int64_t* h00, uint64_t* mcs) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if (replica >= c->R) return kpz_fail(c, KPZ_EINVAL, "replica out of range");
    unsigned long long st[4];
    KPZ_CUDA(c, cudaMemcpyAsync(st, c->d_scratch + c->sl.stats + (size_t)replica * 32, 32, cudaMemcpyDeviceToHost, c->stream));
    KPZ_CUDA(c, cudaStreamSynchronize(c->stream));
    if (attempts) *attempts = c->attempts_base + st[3];
    if (deposits) *deposits = st[0];
    if (removals) *removals = st[1];
    if (h00) *h00 = (int64_t)st[2];
    if (mcs) *mcs = c->mcs;
    return KPZ_OK;
}

int32_t kpz_export_packed(kpz_ctx* c, void* host_dst, size_t bytes) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if (!host_dst || bytes < c->lattice_bytes) return kpz_fail(c, KPZ_EINVAL, "host buffer too small");
    KPZ_CUDA(c, cudaMemcpyAsync(host_dst, c->d_lattice, c->lattice_bytes, cudaMemcpyDeviceToHost, c->stream));
    KPZ_CUDA(c, cudaStreamSynchronize(c->stream));
    return KPZ_OK;
}

int32_t kpz_import_packed(kpz_ctx* c, const void* host_src, size_t bytes, const int64_t* h00, uint64_t mcs) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if (!host_src || bytes < c->lattice_bytes || mcs > 0xFFFFFFFFull) return kpz_fail(c, KPZ_EINVAL, "bad argument");
    KPZ_CUDA(c, cudaMemcpyAsync(c->d_lattice, host_src, c->lattice_bytes, cudaMemcpyHostToDevice, c->stream));
    std::vector<unsigned long long> st((size_t)c->R * 4, 0ull);
    KPZ_CUDA(c, cudaMemcpyAsync(st.data(), c->d_scratch + c->sl.stats, (size_t)c->R * 32, cudaMemcpyDeviceToHost, c->stream));
    KPZ_CUDA(c, cudaStreamSynchronize(c->stream));
    for (uint32_t r = 0; r < c->R; ++r) { st[4 * r + 2] = (unsigned long long)(h00 ? h00[r] : 0); st[4 * r + 3] = 0ull; }
    KPZ_CUDA(c, cudaMemcpyAsync(c->d_scratch + c->sl.stats, st.data(), (size_t)c->R * 32, cudaMemcpyHostToDevice, c->stream));
    KPZ_CUDA(c, cudaStreamSynchronize(c->stream));
    c->mcs = mcs;
    c->attempts_base = mcs * (uint64_t)c->L * c->rows_own;      // rows_own = L for a whole lattice
    return KPZ_OK;
}

int32_t kpz_step_host(kpz_ctx* c, void* host_lattice, size_t bytes, int64_t* h00_inout, uint64_t mcs_start, uint64_t mcs,
                      int64_t* sum_h, int64_t* sum_h2, double* W2) {
    int32_t rc = kpz_import_packed(c, host_lattice, bytes, h00_inout, mcs_start);
    if (rc != KPZ_OK) return rc;
    rc = kpz_run(c, mcs);
    if (rc != KPZ_OK) return rc;
    rc = kpz_measure(c, sum_h, sum_h2, W2);
    if (rc != KPZ_OK && rc != KPZ_EOVERFLOW) return rc;
    int32_t rc2 = kpz_export_packed(c, host_lattice, bytes);
    if (rc2 != KPZ_OK) return rc2;
    if (h00_inout) {
        for (uint32_t r = 0; r < c->R; ++r) {
            int64_t h;
            rc2 = kpz_counters(c, r, nullptr, nullptr, nullptr, &h, nullptr);
            if (rc2 != KPZ_OK) return rc2;
            h00_inout[r] = h;
        }
    }
    return rc;
}

namespace {

// copy streams and events of kpz_pipeline_host: created on the first call, kept in the handle, released by kpz_destroy
int32_t pipeline_resources(kpz_ctx* c, size_t n_events) {
    if (!c->s_in) KPZ_CUDA(c, cudaStreamCreateWithFlags(&c->s_in, cudaStreamNonBlocking));
    if (!c->s_out) KPZ_CUDA(c, cudaStreamCreateWithFlags(&c->s_out, cudaStreamNonBlocking));
    while (c->events.size() < n_events) {
        cudaEvent_t e = nullptr;
        KPZ_CUDA(c, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        c->events.push_back(e);
    }
    return KPZ_OK;
}

// overwrite the tracked h(0,0) of every replica (stats[r][2]) and clear the S7 attempt counter, on the bound stream
int32_t set_h00(kpz_ctx* c, const int64_t* h00) {
    std::vector<unsigned long long> st((size_t)c->R * 4, 0ull);
    KPZ_CUDA(c, cudaMemcpyAsync(st.data(), c->d_scratch + c->sl.stats, (size_t)c->R * 32, cudaMemcpyDeviceToHost, c->stream));
    KPZ_CUDA(c, cudaStreamSynchronize(c->stream));
    for (uint32_t r = 0; r < c->R; ++r) { st[4 * r + 2] = (unsigned long long)(h00 ? h00[r] : 0); st[4 * r + 3] = 0ull; }
    KPZ_CUDA(c, cudaMemcpyAsync(c->d_scratch + c->sl.stats, st.data(), (size_t)c->R * 32, cudaMemcpyHostToDevice, c->stream));
    KPZ_CUDA(c, cudaStreamSynchronize(c->stream));
    return KPZ_OK;
}

// tracked h(0,0) of every replica (stats[r][2]) in one copy on the bound stream
int32_t get_h00(kpz_ctx* c, int64_t* h00) {
    std::vector<unsigned long long> st((size_t)c->R * 4, 0ull);
    KPZ_CUDA(c, cudaMemcpyAsync(st.data(), c->d_scratch + c->sl.stats, (size_t)c->R * 32, cudaMemcpyDeviceToHost, c->stream));
    KPZ_CUDA(c, cudaStreamSynchronize(c->stream));
    for (uint32_t r = 0; r < c->R; ++r) h00[r] = (int64_t)st[4 * r + 2];
    return KPZ_OK;
}

}  // namespace

int32_t kpz_pipeline_host(kpz_ctx* c, void* device_lattice2, size_t device_lattice2_bytes, uint32_t n_lanes,
                          void* const* host_lattices, size_t bytes, int64_t* h00_inout, const uint64_t* mcs_start,
                          uint64_t mcs, uint32_t n_rounds, int64_t* sum_h, int64_t* sum_h2, double* W2) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if ((rc = require_whole(c)) != KPZ_OK) return rc;
    if (!device_lattice2 || device_lattice2_bytes < c->lattice_bytes || ((uintptr_t)device_lattice2 & 15u))
        return kpz_fail(c, KPZ_EINVAL, "second device lattice missing, too small or not 16-byte aligned");
    if (n_lanes == 0 || n_rounds == 0 || !host_lattices || !mcs_start || bytes < c->lattice_bytes)
        return kpz_fail(c, KPZ_EINVAL, "bad argument");
    for (uint32_t l = 0; l < n_lanes; ++l) {
        if (!host_lattices[l]) return kpz_fail(c, KPZ_EINVAL, "NULL host lattice");
        if (mcs_start[l] + (uint64_t)n_rounds * mcs > 0xFFFFFFFFull) return kpz_fail(c, KPZ_EINVAL, "MCS clock would exceed 2^32-1");
    }
    const uint64_t B = (uint64_t)n_lanes * n_rounds;   // batches, b = round * n_lanes + lane
    // per batch two events (copied in, copied out); events are reused round-robin: a batch only ever waits for
    // batches at most max(2, n_lanes) behind it, so a window of that many (+2) batches suffices
    const uint64_t EW = (n_lanes > 2 ? n_lanes : 2) + 2;     // batches in the event window
    rc = pipeline_resources(c, (size_t)EW * 2);
    if (rc != KPZ_OK) return rc;
    struct { cudaStream_t s_in, s_out; cudaEvent_t* ev; uint64_t EW; cudaEvent_t& in(uint64_t b) { return ev[2 * (b % EW)]; }
             cudaEvent_t& out(uint64_t b) { return ev[2 * (b % EW) + 1]; } } res{c->s_in, c->s_out, c->events.data(), EW};
    uint32_t* const dbuf[2] = {c->d_lattice, static_cast<uint32_t*>(device_lattice2)};
    std::vector<int64_t> h00((size_t)n_lanes * c->R, 0);
    if (h00_inout) std::memcpy(h00.data(), h00_inout, h00.size() * sizeof(int64_t));
    std::vector<uint64_t> clock(mcs_start, mcs_start + n_lanes);

    // host->device copy of batch b: its device slot must have been copied out (batch b-2), and so must the last
    // batch of the same lane (b - n_lanes), whose output is this batch's input
    auto enqueue_in = [&](uint64_t b) -> int32_t {
        if (b >= 2) KPZ_CUDA(c, cudaStreamWaitEvent(res.s_in, res.out(b - 2), 0));
        if (b >= n_lanes) KPZ_CUDA(c, cudaStreamWaitEvent(res.s_in, res.out(b - n_lanes), 0));
        KPZ_CUDA(c, cudaMemcpyAsync(dbuf[b & 1], host_lattices[b % n_lanes], c->lattice_bytes, cudaMemcpyHostToDevice, res.s_in));
        KPZ_CUDA(c, cudaEventRecord(res.in(b), res.s_in));
        return KPZ_OK;
    };

    // Order of the host calls in one iteration: every small copy of the bookkeeping (counters out, h(0,0) of the
    // next batch in) is issued while both copy engines are idle, i.e. before the two 'lattice_bytes' copies that
    // follow the kernels; a small copy queued behind one of those would stall the bound stream for its length.
    int32_t worst = KPZ_OK;
    auto body = [&]() -> int32_t {
        int32_t r = set_h00(c, &h00[0]);
        if (r != KPZ_OK) return r;
        if ((r = enqueue_in(0)) != KPZ_OK) return r;
        for (uint64_t b = 0; b < B; ++b) {
            const uint32_t lane = (uint32_t)(b % n_lanes);
            // with one lane the next input is this batch's output: nothing to overlap, copy in after copy out
            if (n_lanes >= 2 && b + 1 < B && (r = enqueue_in(b + 1)) != KPZ_OK) return r;
            c->d_lattice = dbuf[b & 1];
            c->mcs = clock[lane];
            c->attempts_base = clock[lane] * (uint64_t)c->L * c->L;
            KPZ_CUDA(c, cudaStreamWaitEvent(c->stream, res.in(b), 0));
            if ((r = kpz_run(c, mcs)) != KPZ_OK) return r;
            const size_t o = (size_t)b * c->R;
            r = kpz_measure(c, sum_h ? sum_h + o : nullptr, sum_h2 ? sum_h2 + o : nullptr, W2 ? W2 + o : nullptr);
            if (r == KPZ_EOVERFLOW) worst = r;
            else if (r != KPZ_OK) return r;
            // kpz_measure synchronised the bound stream: the lattice of batch b is final
            if ((r = get_h00(c, &h00[(size_t)lane * c->R])) != KPZ_OK) return r;
            clock[lane] += mcs;
            if (b + 1 < B && (r = set_h00(c, &h00[(size_t)((b + 1) % n_lanes) * c->R])) != KPZ_OK) return r;
            KPZ_CUDA(c, cudaMemcpyAsync(host_lattices[lane], dbuf[b & 1], c->lattice_bytes, cudaMemcpyDeviceToHost, res.s_out));
            KPZ_CUDA(c, cudaEventRecord(res.out(b), res.s_out));
            if (n_lanes == 1 && b + 1 < B && (r = enqueue_in(b + 1)) != KPZ_OK) return r;
        }
        KPZ_CUDA(c, cudaStreamSynchronize(res.s_out));
        return KPZ_OK;
    };
    rc = body();
    c->d_lattice = dbuf[0];
    if (rc != KPZ_OK) {          // drain the copy streams before their buffers can go away
        cudaStreamSynchronize(res.s_in);
        cudaStreamSynchronize(res.s_out);
        return rc;
    }
    if (h00_inout) std::memcpy(h00_inout, h00.data(), h00.size() * sizeof(int64_t));
    return worst;
}

// ---- kpz_step_host_overlapped: one lattice, copies overlapped with the kernels slab by slab -------------------------
// A colour pass of a tile touches only the T + 1 storage rows of its footprint, so dependencies between passes spread
// by at most T + 1 rows per pass.  The lattice is cut into n_slabs blocks of rows that arrive one after the other.
// After block s has arrived, stage s runs ALL P = 4 mcs passes, pass p on the tiles whose footprint lies inside
//   [ g_p , f_{s,p} ],   g_p = p (T + 1),   f_{s,p} = (last arrived row) - p (T + 1),
// (the blocks are small at both ends and large in the middle, see below)
// and that no earlier stage has processed: every earlier-pass tile that meets such a footprint lies inside the region
// of an earlier pass of a stage <= s, hence was launched before.  The last stage takes everything that is left (the
// wedges below g_p and above the last frontier, including the tile row that wraps around the lattice edge), again in
// pass order.  Rows that no later tile can touch are copied back while later stages still compute.  Same kernels, same
// tile ids, same streams as kpz_run: the trajectory is bit-identical (tests/test_gpu_parity.py).
namespace {

inline long long floor_div(long long a, long long b) { return a >= 0 ? a / b : -((-a + b - 1) / b); }
inline long long ceil_div(long long a, long long b) { return -floor_div(-a, b); }

// launches colour pass `slot` of MCS m on the tile rows [a, b] (frame of MCS m; b may exceed NT - 1: wrapped range)
int32_t launch_pass_rows(kpz_ctx* c, uint32_t m, uint32_t slot, uint32_t cy, long long a, long long b) {
    if (b < a) return KPZ_OK;
    const long long jf = a > (long long)cy ? (a - cy + 1) / 2 : 0;       // ceil((a - cy) / 2), >= 0
    if (b < (long long)cy) return KPZ_OK;
    const long long jl = (b - cy) / 2;
    if (jl < jf) return KPZ_OK;
    kpz::UpdateParams P;
    fill_update_params(c, P, m, slot, 0u);
    P.j0 = (uint32_t)jf;
    P.HNy = (uint32_t)(jl - jf + 1);
    P.tiles_per_colour = P.HN * P.HNy;
    P.total_items = (uint64_t)P.tiles_per_colour;
    P.blocked = (P.HN % 8 == 0 && P.HNy % 4 == 0) ? 1u : 0u;
    return c->T >= 32 ? kpz_launch_update_wide(c, P) : kpz_launch_update_narrow(c, P);
}

// The schedule of kpz_step_host_overlapped as plain host data (no CUDA): row boundaries of the blocks, the launches in
// issue order (stage, pass, tile rows [a, b] of the frame of that pass's MCS, b may exceed NT - 1: wrapped range; the
// colour of the pass then picks every second row), and the rows that may be copied back after each stage.
// oy[m] = y offset of the global draw of the m-th MCS of the step.  False: the shape does not allow the overlap.
struct OverlapLaunch { uint32_t stage, pass; long long a, b; };
struct OverlapCopy { uint32_t stage; long long r0, r1; };
struct OverlapPlan {
    std::vector<long long> B;
    std::vector<OverlapLaunch> launches;
    std::vector<OverlapCopy> copies;
};

bool overlap_plan(long long L, long long T, long long mcs, long long n_slabs, long long wave_tiles, const uint32_t* oy,
                  OverlapPlan& pl) {
    pl.B.clear();
    pl.launches.clear();
    pl.copies.clear();
    if (mcs < 1 || n_slabs < 2 || T < 1 || L % (2 * T) != 0) return false;
    const long long NT = L / T, P_ = 4 * mcs, step = T + 1;
    // Block heights: compute is the bottleneck (the kernels of a step take about three times its copies), so only the
    // FIRST copy-in and the LAST copy-out are exposed: the blocks ramp up geometrically (x2) from both ends and are
    // large in the middle (few launches, little tail).  Every block must be taller than C_min.
    const long long C_min = 2 * P_ * step + 4 * T;
    bool eligible = false;
    // (a) whole waves: a launch of a middle stage covers (block height / 2T) tile rows of its colour, L / 2T tiles each;
    // the GPU holds wave_tiles tiles at a time, so a block of k waves minus a bit wastes nothing in the last wave of its
    // 4 mcs launches.  Blocks of kmin, 2 kmin, 4 kmin .. waves from both ends, the middle block takes the rest.
    const double q = wave_tiles > 0 ? (double)wave_tiles / (double)(L / (2 * T)) : 0.0;      // colour rows per wave
    if (q >= 1.0) {
        auto rows_for = [&](long long k) { return (long long)std::floor((double)k * q) * 2 * T; };
        long long kmin = 1;
        while (rows_for(kmin) < C_min) ++kmin;
        for (long long S_try = n_slabs; S_try >= 3 && !eligible; --S_try) {
            const long long mid = S_try / 2;
            std::vector<long long> h((size_t)S_try, 0);
            long long sum = 0;
            for (long long i = 0; i < S_try; ++i) {
                if (i == mid) continue;
                const long long e = std::min(i, S_try - 1 - i);
                h[(size_t)i] = rows_for(kmin << std::min<long long>(e, 20));
                sum += h[(size_t)i];
            }
            h[(size_t)mid] = L - sum;
            if (h[(size_t)mid] < C_min) continue;
            pl.B.assign(1, 0);
            for (long long i = 0; i < S_try; ++i) pl.B.push_back(pl.B.back() + h[(size_t)i]);
            eligible = true;
        }
    }
    // (b) otherwise in proportion 1 : 2 : 4 .. : 4 : 2 : 1
    for (long long S_try = n_slabs; S_try >= 2 && !eligible; --S_try) {
        std::vector<long long> w((size_t)S_try);
        long long wsum = 0;
        for (long long i = 0; i < S_try; ++i) {
            const long long e = std::min(i, S_try - 1 - i);
            w[(size_t)i] = 1ll << std::min<long long>(e, 20);
            wsum += w[(size_t)i];
        }
        pl.B.assign(1, 0);
        long long acc = 0;
        bool ok = true;
        for (long long i = 0; i < S_try; ++i) {
            acc += w[(size_t)i];
            const long long b = (i == S_try - 1) ? L : (L * acc / wsum) / (2 * T) * (2 * T);     // whole tile-row pairs
            if (b - pl.B.back() < C_min) { ok = false; break; }
            pl.B.push_back(b);
        }
        eligible = ok;
    }
    if (!eligible) { pl.B.clear(); return false; }
    const std::vector<long long>& B = pl.B;
    const long long S = (long long)B.size() - 1;
    const long long g_last = (P_ - 1) * step;                               // g_{P-1}
    long long out_next = g_last + T;                                        // first row not yet copied back
    for (long long s = 0; s < S; ++s) {
        for (long long p = 0; p < P_; ++p) {
            const long long o = (long long)oy[p / 4];
            const long long g = p * step;
            const long long t_lo = ceil_div(g - o, T) < 0 ? 0 : ceil_div(g - o, T);
            auto t_hi = [&](long long stage) { return floor_div((B[(size_t)stage + 1] - 1 - p * step) - T - o, T); };
            long long a, b;
            if (s < S - 1) {
                a = s == 0 ? t_lo : std::max(t_lo, t_hi(s - 1) + 1);
                b = t_hi(s);
            } else {
                a = std::max(t_lo, t_hi(S - 2) + 1);
                b = NT - 1 + t_lo;                                          // wraps: tile rows 0 .. t_lo - 1 come last
            }
            if (b >= a) pl.launches.push_back({(uint32_t)s, (uint32_t)p, a, b});
        }
        if (s < S - 1) {
            const long long hi = (B[(size_t)s + 1] - 1 - (P_ - 1) * step) - T;  // rows <= f_{s,P-1} - T are final
            if (hi >= out_next) {
                pl.copies.push_back({(uint32_t)s, out_next, hi});
                out_next = hi + 1;
            }
        } else {
            pl.copies.push_back({(uint32_t)s, out_next, L - 1});
            pl.copies.push_back({(uint32_t)s, 0, g_last + T - 1});
        }
    }
    return true;
}

}  // namespace

int32_t kpz_overlap_plan(uint32_t L, uint32_t tile, uint64_t mcs, uint32_t n_slabs, uint32_t wave_tiles, const uint32_t* oy,
                         int64_t* boundaries, uint32_t* n_stages, int64_t* launches, uint32_t* n_launches, int64_t* copies,
                         uint32_t* n_copies) {
    if (!oy || !boundaries || !n_stages || !launches || !n_launches || !copies || !n_copies) return KPZ_EINVAL;
    if (L == 0 || tile == 0 || L % (2 * tile) != 0 || mcs == 0 || mcs > 0xFFFFFFFFull || n_slabs > 4096) return KPZ_EINVAL;
    for (uint64_t m = 0; m < mcs; ++m)
        if (oy[m] >= tile) return KPZ_EINVAL;
    OverlapPlan pl;
    *n_stages = *n_launches = *n_copies = 0;
    if (!overlap_plan(L, tile, (long long)mcs, n_slabs, wave_tiles, oy, pl)) return KPZ_OK;      // no overlap for this shape
    *n_stages = (uint32_t)(pl.B.size() - 1);
    for (size_t i = 0; i < pl.B.size(); ++i) boundaries[i] = pl.B[i];
    *n_launches = (uint32_t)pl.launches.size();
    for (size_t i = 0; i < pl.launches.size(); ++i) {
        launches[4 * i + 0] = pl.launches[i].stage;
        launches[4 * i + 1] = pl.launches[i].pass;
        launches[4 * i + 2] = pl.launches[i].a;
        launches[4 * i + 3] = pl.launches[i].b;
    }
    *n_copies = (uint32_t)pl.copies.size();
    for (size_t i = 0; i < pl.copies.size(); ++i) {
        copies[3 * i + 0] = pl.copies[i].stage;
        copies[3 * i + 1] = pl.copies[i].r0;
        copies[3 * i + 2] = pl.copies[i].r1;
    }
    return KPZ_OK;
}

int32_t kpz_step_host_overlapped(kpz_ctx* c, void* host_lattice, size_t bytes, int64_t* h00_inout, uint64_t mcs_start,
                                 uint64_t mcs, uint32_t n_slabs, int64_t* sum_h, int64_t* sum_h2, double* W2) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if ((rc = require_whole(c)) != KPZ_OK) return rc;
    if (!host_lattice || bytes < c->lattice_bytes || mcs_start + mcs > 0xFFFFFFFFull) return kpz_fail(c, KPZ_EINVAL, "bad argument");
    const long long L = c->L;
    ResidentPlan rp{};
    // the overlap needs: one replica, the default schedule on the tiled kernel, and blocks much taller than the
    // region the passes of the step eat away on both sides (overlap_plan); otherwise the plain sequence (same result)
    OverlapPlan plan;
    std::vector<uint32_t> oy, cy;
    bool eligible = c->R == 1 && c->schedule == KPZ_SCHEDULE_COLOURS && c->sub_sweeps == 1 && !c->poisson && mcs >= 1 &&
                    n_slabs >= 2 && choose_path(c, rp) == KPZ_PATH_TILED;
    if (eligible) {
        oy.resize((size_t)mcs);
        cy.resize((size_t)(4 * mcs));
        for (uint64_t m = 0; m < mcs; ++m) {
            uint32_t ox, oyv, perm[4];
            host_global_draw(c, (uint32_t)(mcs_start + m), 0u, 0u, &ox, &oyv, perm);
            oy[(size_t)m] = oyv;
            for (int slot = 0; slot < 4; ++slot) cy[(size_t)(4 * m) + slot] = perm[slot] >> 1;
        }
        // tiles one wave of the update kernel holds (its CTA shapes: kpz_launch_update_wide.cu): blocks of whole waves
        int sms = 0;
        KPZ_CUDA(c, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, c->device));
        const long long per_sm = c->T == 64 ? 288 : (c->T == 32 ? 512 : 0);
        const long long wave_tiles = (long long)sms * per_sm;
        eligible = overlap_plan(L, c->T, (long long)mcs, n_slabs, wave_tiles, oy.data(), plan);
    }
    if (!eligible) return kpz_step_host(c, host_lattice, bytes, h00_inout, mcs_start, mcs, sum_h, sum_h2, W2);
    const std::vector<long long>& B = plan.B;
    const long long S = (long long)B.size() - 1;
    const size_t row_bytes = (size_t)L / 8, plane_bytes = (size_t)L * row_bytes;
    unsigned char* hb = static_cast<unsigned char*>(host_lattice);
    unsigned char* db = reinterpret_cast<unsigned char*>(c->d_lattice);
    // bookkeeping copies first, while the copy engines are idle
    if ((rc = set_h00(c, h00_inout)) != KPZ_OK) return rc;
    if ((rc = pipeline_resources(c, (size_t)(2 * S + 2))) != KPZ_OK) return rc;
    cudaEvent_t* ev_in = c->events.data();
    cudaEvent_t* ev_cmp = c->events.data() + S;
    c->mcs = mcs_start;
    c->attempts_base = mcs_start * (uint64_t)c->L * c->L;
    // all blocks are queued on the copy-in stream at once: they arrive in order
    for (long long s = 0; s < S; ++s) {
        for (int pln = 0; pln < 2; ++pln) {
            const size_t off = pln * plane_bytes + (size_t)B[(size_t)s] * row_bytes;
            KPZ_CUDA(c, cudaMemcpyAsync(db + off, hb + off, (size_t)(B[(size_t)s + 1] - B[(size_t)s]) * row_bytes,
                                        cudaMemcpyHostToDevice, c->s_in));
        }
        KPZ_CUDA(c, cudaEventRecord(ev_in[s], c->s_in));
    }
    size_t li = 0, ci = 0;
    for (long long s = 0; s < S; ++s) {
        KPZ_CUDA(c, cudaStreamWaitEvent(c->stream, ev_in[s], 0));
        for (; li < plan.launches.size() && plan.launches[li].stage == (uint32_t)s; ++li) {
            const OverlapLaunch& ln = plan.launches[li];
            const uint32_t m = (uint32_t)(mcs_start + (uint64_t)(ln.pass / 4)), slot = ln.pass % 4;
            if ((rc = launch_pass_rows(c, m, slot, cy[ln.pass], ln.a, ln.b)) != KPZ_OK) return rc;
        }
        KPZ_CUDA(c, cudaEventRecord(ev_cmp[s], c->stream));
        KPZ_CUDA(c, cudaStreamWaitEvent(c->s_out, ev_cmp[s], 0));
        for (; ci < plan.copies.size() && plan.copies[ci].stage == (uint32_t)s; ++ci) {
            const OverlapCopy& cp = plan.copies[ci];                         // rows [r0, r1] of both planes
            for (int pln = 0; pln < 2; ++pln) {
                const size_t off = pln * plane_bytes + (size_t)cp.r0 * row_bytes;
                KPZ_CUDA(c, cudaMemcpyAsync(hb + off, db + off, (size_t)(cp.r1 - cp.r0 + 1) * row_bytes, cudaMemcpyDeviceToHost, c->s_out));
            }
        }
    }
    c->mcs = mcs_start + mcs;
    c->attempts_base = c->mcs * (uint64_t)c->L * c->L;
    rc = kpz_measure(c, sum_h, sum_h2, W2);                                 // reads the final lattice while it is copied back
    if (rc != KPZ_OK && rc != KPZ_EOVERFLOW) { cudaStreamSynchronize(c->s_out); return rc; }
    if (h00_inout) {
        const int32_t r2 = get_h00(c, h00_inout);
        if (r2 != KPZ_OK) { cudaStreamSynchronize(c->s_out); return r2; }
    }
    KPZ_CUDA(c, cudaStreamSynchronize(c->s_out));
    return rc;
}

// profiles of replica `replica` relative to h00 on the device (scratch prof[2][L]) + spectra; shared by the two calls
static int32_t run_profiles(kpz_ctx* c, uint32_t replica, bool with_fft, long long* h00_out) {
    const uint32_t L = c->L, W = L / 32;
    uint32_t logL = 0;
    while ((1u << logL) < L) ++logL;
    if (with_fft && (1u << logL) != L) return kpz_fail(c, KPZ_EINVAL, "the power spectrum needs L to be a power of two");
    std::vector<i128> S1, S2;
    std::vector<long long> h00;
    int32_t rc = measure_relative(c, S1, S2, h00, true, replica);
    if (rc != KPZ_OK) return rc;
    *h00_out = h00[replica];
    unsigned char* sc = c->d_scratch;
    const uint64_t plane_words = (uint64_t)L * L / 32;
    int32_t* inc = reinterpret_cast<int32_t*>(sc + c->sl.rowinc);
    kpz::kpz_row_inc_kernel<<<grid_for((uint64_t)L * 32, 256), 256, 0, c->stream>>>(c->d_lattice, plane_words, replica, L, W, inc);
    KPZ_CUDA(c, cudaGetLastError());
    kpz::kpz_profile_fft_kernel<<<2, 1024, 0, c->stream>>>(
        reinterpret_cast<const long long*>(sc + c->sl.colsum), reinterpret_cast<const int32_t*>(sc + c->sl.base) + (size_t)replica * L,
        inc, reinterpret_cast<long long*>(sc + c->sl.prof), reinterpret_cast<double2*>(sc + c->sl.fft),
        reinterpret_cast<double*>(sc + c->sl.sdir), L, with_fft ? logL : 0u);
    KPZ_CUDA(c, cudaGetLastError());
    c->launches += 2;
    if (with_fft) {
        const uint32_t n = L / 2 + 1;
        kpz::kpz_spectrum_average_kernel<<<(n + 255) / 256, 256, 0, c->stream>>>(reinterpret_cast<const double*>(sc + c->sl.sdir),
                                                                           reinterpret_cast<double*>(sc + c->sl.savg), n);
        KPZ_CUDA(c, cudaGetLastError());
        c->launches++;
    }
    return KPZ_OK;
}

int32_t kpz_profiles(kpz_ctx* c, uint32_t replica, int64_t* col_sums, int64_t* row_sums) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if ((rc = require_whole(c)) != KPZ_OK) return rc;
    if (replica >= c->R) return kpz_fail(c, KPZ_EINVAL, "replica out of range");
    long long h00 = 0;
    rc = run_profiles(c, replica, false, &h00);
    if (rc != KPZ_OK) return rc;
    const uint32_t L = c->L;
    std::vector<long long> prof((size_t)2 * L);
    KPZ_CUDA(c, cudaMemcpyAsync(prof.data(), c->d_scratch + c->sl.prof, (size_t)2 * L * 8, cudaMemcpyDeviceToHost, c->stream));
    KPZ_CUDA(c, cudaStreamSynchronize(c->stream));
    for (uint32_t i = 0; i < L; ++i) {
        if (col_sums) col_sums[i] = prof[i] + (long long)L * h00;
        if (row_sums) row_sums[i] = prof[(size_t)L + i] + (long long)L * h00;
    }
    return KPZ_OK;
}

int32_t kpz_power_spectrum(kpz_ctx* c, uint32_t replica, double* S, double* Sx, double* Sy) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if ((rc = require_whole(c)) != KPZ_OK) return rc;
    if (replica >= c->R) return kpz_fail(c, KPZ_EINVAL, "replica out of range");
    long long h00 = 0;
    rc = run_profiles(c, replica, true, &h00);
    if (rc != KPZ_OK) return rc;
    const size_t n = c->L / 2 + 1;
    if (S) KPZ_CUDA(c, cudaMemcpyAsync(S, c->d_scratch + c->sl.savg, n * 8, cudaMemcpyDeviceToHost, c->stream));
    if (Sx) KPZ_CUDA(c, cudaMemcpyAsync(Sx, c->d_scratch + c->sl.sdir, n * 8, cudaMemcpyDeviceToHost, c->stream));
    if (Sy) KPZ_CUDA(c, cudaMemcpyAsync(Sy, c->d_scratch + c->sl.sdir + n * 8, n * 8, cudaMemcpyDeviceToHost, c->stream));
    KPZ_CUDA(c, cudaStreamSynchronize(c->stream));
    return KPZ_OK;
}


// ---- one lattice split into slabs of rows over several handles / GPUs ---------------------

int32_t kpz_slab_workspace_bytes(uint32_t L, uint32_t tile, uint32_t n_slabs, size_t* lattice_bytes, size_t* scratch_bytes) {
    int32_t rc = validate(L, 0.0, 0.0, tile, 1);
    if (rc != KPZ_OK) return rc;
    if (n_slabs == 0 || (L / tile) % (2 * n_slabs) != 0 || (L / n_slabs) % 32 != 0) return KPZ_EINVAL;
    const size_t rows = (size_t)L / n_slabs + tile + 2;
    if (lattice_bytes) *lattice_bytes = 2 * rows * (L / 8);
    if (scratch_bytes) *scratch_bytes = scratch_layout(L, 1).total;
    return KPZ_OK;
}

int32_t kpz_create_slab(kpz_ctx** out, uint32_t L, double p, double q, uint32_t tile, uint64_t seed, uint32_t n_slabs,
                        uint32_t slab) {
    if (!out) return KPZ_EINVAL;
    *out = nullptr;
    size_t lat = 0;
    int32_t rc = kpz_slab_workspace_bytes(L, tile, n_slabs, &lat, nullptr);
    if (rc != KPZ_OK || slab >= n_slabs) return KPZ_EINVAL;
    rc = kpz_create_batch(out, L, p, q, tile, seed, 1);
    if (rc != KPZ_OK) return rc;
    kpz_ctx* c = *out;
    c->n_slabs = n_slabs;
    c->slab = slab;
    c->rows_own = L / n_slabs;
    c->rows = c->rows_own + tile + 2;
    c->lattice_bytes = lat;
    return KPZ_OK;
}

int32_t kpz_slab_info(const kpz_ctx* c, uint32_t* rows_own, uint32_t* rows_stored, size_t* row_bytes, size_t* base_offset,
                      size_t* totals_offset) {
    if (!c || c->n_slabs == 0) return KPZ_EINVAL;
    if (rows_own) *rows_own = c->rows_own;
    if (rows_stored) *rows_stored = c->rows;
    if (row_bytes) *row_bytes = c->L / 8;
    if (base_offset) *base_offset = c->sl.base;
    if (totals_offset) *totals_offset = c->sl.rowinc;
    return KPZ_OK;
}

int32_t kpz_global_draw(const kpz_ctx* c, uint64_t m, uint32_t* ox, uint32_t* oy, uint32_t* perm) {
    if (!c || !ox || !oy || !perm || m > 0xFFFFFFFFull) return KPZ_EINVAL;
    host_global_draw(c, (uint32_t)m, 0u, 0u, ox, oy, perm);
    return KPZ_OK;
}

int32_t kpz_slab_pass(kpz_ctx* c, uint32_t slot) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if (c->n_slabs == 0) return kpz_fail(c, KPZ_ESTATE, "not a slab handle");
    if (slot > 3 || c->schedule != KPZ_SCHEDULE_COLOURS || c->sub_sweeps != 1 || c->poisson)
        return kpz_fail(c, KPZ_EINVAL, "slabs run the default schedule, colour passes 0..3");
    if (c->mcs >= 0xFFFFFFFFull) return kpz_fail(c, KPZ_EINVAL, "MCS clock would exceed 2^32-1");
    return launch_update(c, (uint32_t)c->mcs, slot, 0u);
}

int32_t kpz_slab_end_mcs(kpz_ctx* c) {
    if (!c || c->n_slabs == 0) return KPZ_EINVAL;
    if (c->mcs >= 0xFFFFFFFFull) return kpz_fail(c, KPZ_EINVAL, "MCS clock would exceed 2^32-1");
    c->mcs++;
    c->attempts_base += (uint64_t)c->L * c->rows_own;
    return KPZ_OK;
}

int32_t kpz_slab_measure_local(kpz_ctx* c) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if (c->n_slabs == 0) return kpz_fail(c, KPZ_ESTATE, "not a slab handle");
    const uint32_t L = c->L, W = L / 32;
    const uint64_t plane_words = (uint64_t)c->rows * W;
    unsigned char* sc = c->d_scratch;
    int32_t* base = reinterpret_cast<int32_t*>(sc + c->sl.base);
    int32_t* cS0 = reinterpret_cast<int32_t*>(sc + c->sl.cS0);
    int32_t* cS1 = reinterpret_cast<int32_t*>(sc + c->sl.cS1);
    int32_t* cS2 = reinterpret_cast<int32_t*>(sc + c->sl.cS2);
    if (c->slab == 0) {       // the walk along x on lattice row 0 (eq. 3) lives on slab 0
        int nthr = 1024;
        while (nthr > 32 && (uint32_t)nthr > L) nthr >>= 1;
        kpz::kpz_row0_prefix_kernel<<<1, nthr, 0, c->stream>>>(c->d_lattice, plane_words, L, W, base);
        KPZ_CUDA(c, cudaGetLastError());
        c->launches++;
    }
    dim3 g1((W + 127) / 128, c->sl.n_chunks, 1);
    kpz::kpz_column_chunk_kernel<<<g1, 128, 0, c->stream>>>(c->d_lattice, plane_words, L, W, c->sl.rows_per_chunk, cS0, cS1, cS2,
                                                         c->rows_own, c->slab == 0 ? 1u : 0u);
    KPZ_CUDA(c, cudaGetLastError());
    kpz::kpz_slab_totals_kernel<<<(L + 255) / 256, 256, 0, c->stream>>>(cS0, L, c->sl.n_chunks, c->sl.rows_per_chunk, c->rows_own,
                                                                    reinterpret_cast<int32_t*>(sc + c->sl.rowinc));
    KPZ_CUDA(c, cudaGetLastError());
    c->launches += 2;
    return KPZ_OK;
}

int32_t kpz_slab_measure_finish(kpz_ctx* c, const void* d_base0, const void* d_totals_all, uint64_t* halves) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if (c->n_slabs == 0) return kpz_fail(c, KPZ_ESTATE, "not a slab handle");
    if (!d_base0 || !d_totals_all || !halves) return kpz_fail(c, KPZ_EINVAL, "NULL argument");
    const uint32_t L = c->L;
    unsigned char* sc = c->d_scratch;
    unsigned long long* msum = reinterpret_cast<unsigned long long*>(sc + c->sl.msum);
    KPZ_CUDA(c, cudaMemsetAsync(msum, 0, 32, c->stream));
    // the entry height of this slab's columns; prof (unused on slab handles) holds it so that base0 may alias `base`
    int32_t* mybase = reinterpret_cast<int32_t*>(sc + c->sl.prof);
    kpz::kpz_slab_base_kernel<<<(L + 255) / 256, 256, 0, c->stream>>>(static_cast<const int32_t*>(d_base0),
                                                                  static_cast<const int32_t*>(d_totals_all), L, c->slab, mybase);
    KPZ_CUDA(c, cudaGetLastError());
    dim3 g2((L + 255) / 256, 1);
    kpz::kpz_combine_kernel<<<g2, 256, 0, c->stream>>>(mybase, reinterpret_cast<int32_t*>(sc + c->sl.cS0),
                                                    reinterpret_cast<int32_t*>(sc + c->sl.cS1),
                                                    reinterpret_cast<int32_t*>(sc + c->sl.cS2), L, c->sl.n_chunks,
                                                    c->sl.rows_per_chunk, msum, nullptr, 0u, c->rows_own);
    KPZ_CUDA(c, cudaGetLastError());
    c->launches += 2;
    unsigned long long hm[4];
    KPZ_CUDA(c, cudaMemcpyAsync(hm, msum, 32, cudaMemcpyDeviceToHost, c->stream));
    KPZ_CUDA(c, cudaStreamSynchronize(c->stream));
    for (int k = 0; k < 4; ++k) halves[k] = hm[k];
    return KPZ_OK;
}

int32_t kpz_slab_finalize(uint32_t L, const uint64_t* halves, int64_t h00, int64_t* sum_h, int64_t* sum_h2, double* W2) {
    if (!halves || L == 0) return KPZ_EINVAL;
    // halves: {lo, hi} 32-bit-half accumulators of sum (h - h00) and of sum (h - h00)^2, summed over the slabs
    const i128 S1 = (i128)(long long)halves[1] * ((i128)1 << 32) + (i128)halves[0];
    const i128 S2 = (i128)(long long)halves[3] * ((i128)1 << 32) + (i128)halves[2];
    return finalize_sums(L, S1, S2, (long long)h00, sum_h, sum_h2, W2) ? KPZ_EOVERFLOW : KPZ_OK;
}

int32_t kpz_launch_count(const kpz_ctx* c, uint64_t* out) {
    if (!c || !out) return KPZ_EINVAL;
    *out = c->launches;
    return KPZ_OK;
}

int32_t kpz_measure_peaks(double* out, uint32_t n) {
    if (!out || n < KPZ_N_PEAKS) return KPZ_EINVAL;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return KPZ_ECUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) return KPZ_ECUDA;
    const uint32_t blocks = (uint32_t)sms * 8u;              // 8 CTAs of 256 threads per SM: every warp slot busy
    uint32_t* sink = nullptr;
    unsigned long long* ticks = nullptr;
    if (cudaMalloc(&sink, blocks * sizeof(uint32_t)) != cudaSuccess) { cudaGetLastError(); return KPZ_ECUDA; }
    if (cudaMalloc(&ticks, 16) != cudaSuccess) { cudaGetLastError(); cudaFree(sink); return KPZ_ECUDA; }
    const uint32_t iters = 2048;
    const double lanes = (double)blocks * 256.0 * iters * kpz::PEAK_UNROLL;        // lane-instructions of the measured kind
    float ms[7] = {0, 0, 0, 0, 0, 0, 0};
    cudaError_t e = run_peak<kpz::PEAK_LOP3>(blocks, iters, sink, ticks, &ms[0]);
    unsigned long long hticks[2] = {0, 1};
    if (e == cudaSuccess) e = cudaMemcpy(hticks, ticks, 16, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = run_peak<kpz::PEAK_SHF>(blocks, iters, sink, ticks, &ms[1]);
    if (e == cudaSuccess) e = run_peak<kpz::PEAK_IMAD>(blocks, iters, sink, ticks, &ms[2]);
    if (e == cudaSuccess) e = run_peak<kpz::PEAK_IMAD_WIDE>(blocks, iters, sink, ticks, &ms[3]);
    if (e == cudaSuccess) e = run_peak<kpz::PEAK_LDS>(blocks, iters, sink, ticks, &ms[4]);
    if (e == cudaSuccess) e = run_peak<kpz::PEAK_ATOMS>(blocks, iters, sink, ticks, &ms[5]);
    if (e == cudaSuccess) e = run_peak<kpz::PEAK_MIX>(blocks, iters / 4, sink, ticks, &ms[6]);
    // the dependent chain of one tile: 1 and 2 warps per scheduler on one SM
    unsigned long long cticks[2] = {0, 0};
    for (int v = 0; v < 2 && e == cudaSuccess; ++v) {
        const uint32_t citers = 50000;
        kpz::kpz_chain_kernel<<<1, v == 0 ? 128 : 256>>>(citers, 1234u, ticks);
        e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaMemcpy(&cticks[v], ticks, 8, cudaMemcpyDeviceToHost);
        out[9 + v] = (double)cticks[v] / citers;
    }
    cudaFree(sink);
    cudaFree(ticks);
    if (e != cudaSuccess) return KPZ_ECUDA;
    out[0] = (double)hticks[0] / ((double)(hticks[1] ? hticks[1] : 1) * 1e-9);   // SM clock while the LOP3 kernel ran
    out[1] = lanes / (ms[0] * 1e-3);                   // LOP3 lane-ops/s
    out[2] = lanes / (ms[1] * 1e-3);                   // SHF lane-ops/s
    out[3] = lanes / (ms[2] * 1e-3);                   // IMAD lane-ops/s
    out[4] = lanes / (ms[3] * 1e-3);                   // IMAD.WIDE lane-ops/s (one LOP3 rides along each)
    out[5] = lanes * 4.0 / (ms[4] * 1e-3);             // LDS.32 bytes/s, every lane in its own bank
    out[6] = lanes / (ms[5] * 1e-3);                   // shared-memory XOR reductions (lane-ops/s)
    out[7] = lanes / 4.0 / (ms[6] * 1e-3);             // attempts/s of the bare instruction mix of one p = 1 attempt, no chain
    out[8] = (double)sms;
    return KPZ_OK;
}

int32_t kpz_measure_layouts(double* out, uint32_t n) {
    if (!out || n < KPZ_N_LAYOUTS) return KPZ_EINVAL;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return KPZ_ECUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) return KPZ_ECUDA;
    uint32_t* sink = nullptr;
    if (cudaMalloc(&sink, sizeof(uint32_t)) != cudaSuccess) { cudaGetLastError(); return KPZ_ECUDA; }
    cudaError_t e = run_layout<0>(sms, sink, &out[0], &out[1]);
    if (e == cudaSuccess) e = run_layout<1>(sms, sink, &out[2], &out[3]);
    cudaFree(sink);
    if (e != cudaSuccess) { cudaGetLastError(); return KPZ_ECUDA; }
    return KPZ_OK;
}

int32_t kpz_philox_selftest(const uint32_t* ctr, const uint32_t* key, uint32_t* out, uint32_t n) {
    if (!ctr || !key || !out || n == 0) return KPZ_EINVAL;
    uint32_t *dc = nullptr, *dk = nullptr, *dout = nullptr;
    if (cudaMalloc(&dc, 16 * (size_t)n) != cudaSuccess) { cudaGetLastError(); return KPZ_ECUDA; }
    if (cudaMalloc(&dk, 8 * (size_t)n) != cudaSuccess) { cudaGetLastError(); cudaFree(dc); return KPZ_ECUDA; }
    if (cudaMalloc(&dout, 16 * (size_t)n) != cudaSuccess) { cudaGetLastError(); cudaFree(dc); cudaFree(dk); return KPZ_ECUDA; }
    cudaError_t e = cudaMemcpy(dc, ctr, 16 * (size_t)n, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(dk, key, 8 * (size_t)n, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        kpz::kpz_philox_selftest_kernel<<<(n + 127) / 128, 128>>>(dc, dk, dout, n);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(out, dout, 16 * (size_t)n, cudaMemcpyDeviceToHost);
    cudaFree(dc); cudaFree(dk); cudaFree(dout);
    return e == cudaSuccess ? KPZ_OK : KPZ_ECUDA;
}

}  // extern "C"
