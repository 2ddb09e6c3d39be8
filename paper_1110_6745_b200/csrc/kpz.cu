// kpz.cu -- host side of libkpz_b200.so: the C ABI of include/kpz.h on top of the kernels in kpz_device.cuh.
// No CPU fallback: every entry point that computes launches CUDA kernels on the bound stream.
#include "../../include/kpz.h"

#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <vector>

#include "kpz_device.cuh"
#include "kpz_resident.cuh"

namespace {

typedef __int128 i128;
typedef unsigned __int128 u128;

struct ScratchLayout {
    size_t stats;     // [R][4] u64 : deposits, removals, h00, reserved
    size_t msum;      // [R][4] u64 : lo/hi halves of sum rel, sum rel^2
    size_t misc;      // 8 x u64    : [0] hash accumulator, [1] validation flags
    size_t base;      // [R][L] i32
    size_t cS0;       // [R][NC][L] i32
    size_t cS1;       // [R][NC][L] i32
    size_t cS2;       // [R][NC][L] i32
    size_t colsum;    // [L] i64       column sums of one replica (power spectrum / profiles)
    size_t rowinc;    // [L] i32
    size_t prof;      // [2][L] i64    column and row profiles relative to h00
    size_t fft;       // [2][L] double2
    size_t sdir;      // [2][L/2+1] double
    size_t savg;      // [L/2+1] double
    size_t ptab;      // [4096] u64     S7 count table
    size_t total;
    uint32_t n_chunks, rows_per_chunk;
};

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

struct kpz_ctx {
    uint32_t L, T, R;
    double p, q;
    uint64_t seed;
    uint64_t mcs;            // completed MCS (all replicas advance together)
    uint64_t launches;
    int32_t schedule;        // KPZ_SCHEDULE_COLOURS or KPZ_SCHEDULE_DEAD_BORDER
    uint32_t sub_sweeps;     // K sub-sweeps per MCS (S6)
    bool poisson;            // Poissonised steps per tile and sub-sweep (S7)
    int32_t path;            // KPZ_PATH_*: which update kernels kpz_run uses
    uint32_t pn, pk_min;     // count table on the device (scratch ptab): entries, smallest count
    uint64_t attempts_base;  // attempts made by fixed-count MCS (S7 MCS count theirs on the device, stats[3])
    uint32_t* d_lattice;
    unsigned char* d_scratch;
    cudaStream_t stream;
    bool bound;
    ScratchLayout sl;
    size_t lattice_bytes;
    int device;              // ordinal of the device that holds the bound buffers (-1 before kpz_bind)
    char err[512];
};

namespace {

int32_t fail(kpz_ctx* c, int32_t code, const char* fmt, ...) {
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof(c->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

#define KPZ_CUDA(c, expr)                                                                          \
    do {                                                                                           \
        cudaError_t e__ = (expr);                                                                  \
        if (e__ != cudaSuccess)                                                                    \
            return fail((c), KPZ_ECUDA, "%s failed: %s", #expr, cudaGetErrorString(e__));          \
    } while (0)

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

constexpr int KPZ_MAX_DEVICES = 64;

int grid_for(uint64_t n, int block, int cap = 148 * 16) {
    uint64_t g = (n + block - 1) / block;
    if (g > (uint64_t)cap) g = cap;
    if (g < 1) g = 1;
    return (int)g;
}

template <int T, int NTHR, int MODE, bool DEAD, int SUB>
int32_t launch_update_k(kpz_ctx* c, const kpz::UpdateParams& P) {
    const size_t smem = (size_t)kpz::TileGeom<T>::WORDS * NTHR * sizeof(uint32_t);
    auto kern = kpz::kpz_update_kernel<T, NTHR, MODE, DEAD, SUB>;
    // function attributes are per device: one flag per device ordinal and instantiation
    static bool attr_set[KPZ_MAX_DEVICES] = {};
    const int dev = (c->device >= 0 && c->device < KPZ_MAX_DEVICES) ? c->device : 0;
    if (!attr_set[dev]) {
        KPZ_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        KPZ_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, 100));
        attr_set[dev] = true;
    }
    const uint64_t blocks = (P.total_items + NTHR - 1) / NTHR;
    if (blocks > 0x7FFFFFFFull) return fail(c, KPZ_EINVAL, "too many tiles for one launch");
    kern<<<(unsigned)blocks, NTHR, smem, c->stream>>>(P);
    KPZ_CUDA(c, cudaGetLastError());
    c->launches++;
    return KPZ_OK;
}

template <int T, int NTHR, int MODE, bool DEAD>
int32_t launch_update_t(kpz_ctx* c, const kpz::UpdateParams& P) {
    if (c->poisson) return launch_update_k<T, NTHR, MODE, DEAD, 2>(c, P);
    return c->sub_sweeps > 1 ? launch_update_k<T, NTHR, MODE, DEAD, 1>(c, P) : launch_update_k<T, NTHR, MODE, DEAD, 0>(c, P);
}

template <int T, int NTHR, bool DEAD>
int32_t launch_update_sched(kpz_ctx* c, const kpz::UpdateParams& P) {
    if (c->p >= 1.0 && c->q <= 0.0) return launch_update_t<T, NTHR, 0, DEAD>(c, P);
    if (P.thr_p >= 1 && P.thr_q >= 1) return launch_update_t<T, NTHR, 1, DEAD>(c, P);
    return launch_update_t<T, NTHR, 2, DEAD>(c, P);
}

template <int T, int NTHR>
int32_t launch_update_mode(kpz_ctx* c, const kpz::UpdateParams& P) {
    return c->schedule == KPZ_SCHEDULE_DEAD_BORDER ? launch_update_sched<T, NTHR, true>(c, P)
                                                   : launch_update_sched<T, NTHR, false>(c, P);
}

int32_t launch_update(kpz_ctx* c, uint32_t m, uint32_t slot, uint32_t sub) {
    kpz::UpdateParams P;
    P.lattice = c->d_lattice;
    P.stats = reinterpret_cast<unsigned long long*>(c->d_scratch + c->sl.stats);
    P.plane_words = (uint64_t)c->L * c->L / 32;
    P.L = c->L;
    P.NT = c->L / c->T;
    P.HN = (c->schedule == KPZ_SCHEDULE_DEAD_BORDER) ? P.NT : P.NT / 2;   // tiles per edge in one launch
    P.W = c->L / 32;
    P.tiles_per_colour = P.HN * P.HN;
    P.total_items = (uint64_t)c->R * P.tiles_per_colour;
    P.blocked = (P.HN % 8 == 0) ? 1u : 0u;
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
    switch (c->T) {
        case 64: return launch_update_mode<64, 96>(c, P);
        case 32: return launch_update_mode<32, 64>(c, P);
        case 16: return launch_update_mode<16, 128>(c, P);
        case 8: return launch_update_mode<8, 128>(c, P);
        case 4: return launch_update_mode<4, 128>(c, P);
    }
    return fail(c, KPZ_EINVAL, "unsupported tile %u", c->T);
}

// ---- lattice-resident path (kpz_resident.cuh): one launch for all `n` MCS ------------------------------------
struct ResidentPlan {
    bool ok;            // the lattice fits and the schedule is the default one
    bool coop;          // one warp per tile (few tiles) instead of one thread per tile
    uint32_t G, threads, blocks;
    size_t smem;
};

constexpr size_t KPZ_RESIDENT_SMEM_MAX = 200 * 1024;

ResidentPlan resident_plan(const kpz_ctx* c, bool coop) {
    ResidentPlan pl{};
    const uint32_t L = c->L, T = c->T;
    const bool general = !(c->p >= 1.0 && c->q <= 0.0);
    const size_t lat = (size_t)L * L / 8;                    // bytes of height bits per replica
    const uint32_t HN = L / T / 2, tpc = HN * HN;
    pl.coop = coop;
    pl.ok = (L & (L - 1)) == 0 && c->schedule == KPZ_SCHEDULE_COLOURS && c->sub_sweeps == 1 && !c->poisson;
    if (!pl.ok) return pl;
    if (coop) {
        const uint32_t nwarps = tpc < 32u ? tpc : 32u;
        pl.G = 1;
        pl.threads = 32u * nwarps;
        pl.blocks = c->R;
        pl.smem = (general ? 3 : 2) * lat + (size_t)nwarps * kpz::KPZ_COOP_WARP_WORDS * 4;
    } else {
        uint32_t G = tpc >= 32u ? 1u : (32u + tpc - 1u) / tpc;     // fill at least one warp
        if (G > c->R) G = c->R;
        while (G > 1 && G * lat > KPZ_RESIDENT_SMEM_MAX) --G;
        const uint64_t items = (uint64_t)G * tpc;
        pl.G = G;
        pl.threads = (uint32_t)(items > 1024 ? 1024 : (items + 31) / 32 * 32);
        pl.blocks = (c->R + G - 1) / G;
        pl.smem = G * lat;
    }
    pl.ok = pl.smem <= KPZ_RESIDENT_SMEM_MAX;
    return pl;
}

template <int T, bool GENERAL, bool COOP>
int32_t launch_resident_k(kpz_ctx* c, const kpz::ResidentParams& P, const ResidentPlan& pl) {
    auto kern = kpz::kpz_resident_kernel<T, GENERAL, COOP>;
    static bool attr_set[KPZ_MAX_DEVICES] = {};
    const int dev = (c->device >= 0 && c->device < KPZ_MAX_DEVICES) ? c->device : 0;
    if (!attr_set[dev]) {
        KPZ_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)KPZ_RESIDENT_SMEM_MAX));
        attr_set[dev] = true;
    }
    kern<<<pl.blocks, pl.threads, pl.smem, c->stream>>>(P);
    KPZ_CUDA(c, cudaGetLastError());
    c->launches++;
    return KPZ_OK;
}

template <int T>
int32_t launch_resident_t(kpz_ctx* c, const kpz::ResidentParams& P, const ResidentPlan& pl) {
    const bool general = !(c->p >= 1.0 && c->q <= 0.0);
    if (pl.coop) return general ? launch_resident_k<T, true, true>(c, P, pl) : launch_resident_k<T, false, true>(c, P, pl);
    return general ? launch_resident_k<T, true, false>(c, P, pl) : launch_resident_k<T, false, false>(c, P, pl);
}

int32_t launch_resident(kpz_ctx* c, const ResidentPlan& pl, uint32_t m0, uint32_t n_mcs) {
    kpz::ResidentParams P;
    P.lattice = c->d_lattice;
    P.stats = reinterpret_cast<unsigned long long*>(c->d_scratch + c->sl.stats);
    P.plane_words = (uint64_t)c->L * c->L / 32;
    P.thr_p = accept_threshold(c->p);
    P.thr_q = accept_threshold(c->q);
    P.L = c->L; P.W = c->L / 32; P.NT = c->L / c->T; P.HN = P.NT / 2; P.tpc = P.HN * P.HN;
    P.R = c->R; P.G = pl.G; P.m0 = m0; P.n_mcs = n_mcs;
    P.key.k0 = (uint32_t)(c->seed & 0xFFFFFFFFull);
    P.key.k1 = (uint32_t)(c->seed >> 32);
    switch (c->T) {
        case 64: return launch_resident_t<64>(c, P, pl);
        case 32: return launch_resident_t<32>(c, P, pl);
        case 16: return launch_resident_t<16>(c, P, pl);
        case 8: return launch_resident_t<8>(c, P, pl);
        case 4: return launch_resident_t<4>(c, P, pl);
    }
    return fail(c, KPZ_EINVAL, "unsupported tile %u", c->T);
}

// Which kernels advance the lattice.  AUTO: the resident kernels when the lattice fits in shared memory and at most
// L = 512 -- one warp per tile when the whole handle has few tiles per colour (a chain-bound lattice), one thread
// per tile otherwise -- else the tiled kernel.
int32_t choose_path(kpz_ctx* c, ResidentPlan& pl) {
    const uint64_t tpc = (uint64_t)(c->L / c->T / 2) * (c->L / c->T / 2);
    if (c->path == KPZ_PATH_TILED) return KPZ_PATH_TILED;
    if (c->path == KPZ_PATH_RESIDENT || c->path == KPZ_PATH_RESIDENT_COOP) {
        pl = resident_plan(c, c->path == KPZ_PATH_RESIDENT_COOP);
        return pl.ok ? c->path : -1;
    }
    if (c->L > 512) return KPZ_PATH_TILED;
    const bool coop = (uint64_t)c->R * tpc <= 2048;
    pl = resident_plan(c, coop);
    if (pl.ok) return coop ? KPZ_PATH_RESIDENT_COOP : KPZ_PATH_RESIDENT;
    return KPZ_PATH_TILED;
}

int32_t require_bound(kpz_ctx* c) {
    if (!c) return KPZ_EINVAL;
    if (!c->bound) return fail(c, KPZ_ESTATE, "kpz_bind has not been called");
    return KPZ_OK;
}

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
                                                         cS1, cS2);
    KPZ_CUDA(c, cudaGetLastError());
    dim3 g2((L + 255) / 256, R);
    kpz::kpz_combine_kernel<<<g2, 256, 0, c->stream>>>(base, cS0, cS1, cS2, L, c->sl.n_chunks, c->sl.rows_per_chunk, msum,
                                                    want_colsum ? reinterpret_cast<long long*>(sc + c->sl.colsum) : nullptr,
                                                    colsum_replica);
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
    c->d_lattice = nullptr; c->d_scratch = nullptr; c->stream = nullptr; c->bound = false; c->device = -1;
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
    if (!d_lattice || !d_scratch) return fail(c, KPZ_EINVAL, "NULL device buffer");
    if (lattice_bytes < c->lattice_bytes || scratch_bytes < c->sl.total)
        return fail(c, KPZ_ENOMEM, "bound buffers too small: need %zu + %zu bytes", c->lattice_bytes, c->sl.total);
    if (((uintptr_t)d_lattice & 15u) || ((uintptr_t)d_scratch & 15u)) return fail(c, KPZ_EINVAL, "buffers must be 16-byte aligned");
    // the device is the one that owns the buffers, whatever device is current in the calling thread
    cudaPointerAttributes al, as;
    KPZ_CUDA(c, cudaPointerGetAttributes(&al, d_lattice));
    KPZ_CUDA(c, cudaPointerGetAttributes(&as, d_scratch));
    if (al.type != cudaMemoryTypeDevice || as.type != cudaMemoryTypeDevice || al.device != as.device)
        return fail(c, KPZ_EINVAL, "lattice and scratch must be device memory of one device");
    if (al.device < 0 || al.device >= KPZ_MAX_DEVICES) return fail(c, KPZ_EINVAL, "device ordinal out of range");
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
    const uint64_t n_words = (uint64_t)c->R * ((uint64_t)c->L * c->L / 16);
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
    if (c->mcs + mcs > 0xFFFFFFFFull) return fail(c, KPZ_EINVAL, "MCS clock would exceed 2^32-1");
    if (mcs == 0) return KPZ_OK;
    ResidentPlan pl{};
    const int32_t path = choose_path(c, pl);
    if (path < 0) return fail(c, KPZ_EINVAL, "the resident path needs a power-of-two L that fits in shared memory and the default schedule");
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
    if (path < KPZ_PATH_AUTO || path > KPZ_PATH_RESIDENT_COOP) return fail(c, KPZ_EINVAL, "unknown path");
    c->path = path;
    return KPZ_OK;
}

int32_t kpz_set_schedule(kpz_ctx* c, int32_t schedule) {
    if (!c) return KPZ_EINVAL;
    if (schedule != KPZ_SCHEDULE_COLOURS && schedule != KPZ_SCHEDULE_DEAD_BORDER) return fail(c, KPZ_EINVAL, "unknown schedule");
    c->schedule = schedule;
    return KPZ_OK;
}

static int32_t upload_poisson_table(kpz_ctx* c);

int32_t kpz_set_sub_sweeps(kpz_ctx* c, uint32_t K) {
    if (!c) return KPZ_EINVAL;
    const uint32_t calls = c->T * c->T / 8u;
    if (K < 1 || K > calls || calls % K != 0) return fail(c, KPZ_EINVAL, "sub-sweeps must divide tile*tile/8");
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
    if (n > 4096) return fail(c, KPZ_EINVAL, "Poisson table too large");
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
    c->poisson = on != 0;
    return c->poisson ? upload_poisson_table(c) : KPZ_OK;
}

int32_t kpz_measure(kpz_ctx* c, int64_t* sum_h, int64_t* sum_h2, double* W2) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    std::vector<i128> S1, S2;
    std::vector<long long> h00;
    rc = measure_relative(c, S1, S2, h00);
    if (rc != KPZ_OK) return rc;
    const i128 N = (i128)c->L * c->L;
    const double Nd = (double)((uint64_t)c->L * c->L);
    bool overflow = false;
    for (uint32_t r = 0; r < c->R; ++r) {
        const i128 h0 = h00[r];
        const i128 sh = S1[r] + N * h0;                          // sum h
        const i128 sh2 = S2[r] + 2 * h0 * S1[r] + N * h0 * h0;   // sum h^2
        // N*sum_h2 - sum_h^2 is invariant under the shift by h0: evaluate it on the small relative sums
        const i128 num = N * S2[r] - S1[r] * S1[r];
        if (W2) W2[r] = (double)num / (Nd * Nd);
        if (sum_h) { if (fits_i64(sh)) sum_h[r] = (int64_t)sh; else { sum_h[r] = 0; overflow = true; } }
        if (sum_h2) { if (fits_i64(sh2)) sum_h2[r] = (int64_t)sh2; else { sum_h2[r] = 0; overflow = true; } }
    }
    if (overflow) return fail(c, KPZ_EOVERFLOW, "a sum does not fit int64");
    return KPZ_OK;
}

int32_t kpz_run_sampled(kpz_ctx* c, const uint64_t* times, uint32_t n_times, int64_t* sum_h, int64_t* sum_h2, double* W2) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if (!times || n_times == 0) return fail(c, KPZ_EINVAL, "no sampling times");
    uint64_t prev = c->mcs;
    for (uint32_t i = 0; i < n_times; ++i) {
        if (times[i] < prev || (i > 0 && times[i] == times[i - 1])) return fail(c, KPZ_EINVAL, "sampling times must increase from the current MCS clock");
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
    if (replica >= c->R || !sx || !sy || w == 0 || h == 0 || w > c->L || h > c->L) return fail(c, KPZ_EINVAL, "bad window");
    const size_t n = (size_t)w * h;
    int8_t* d = nullptr;
    if (cudaMalloc(&d, 2 * n) != cudaSuccess) { cudaGetLastError(); return fail(c, KPZ_ENOMEM, "temporary device buffer"); }
    kpz::kpz_unpack_window_kernel<<<grid_for(n, 256), 256, 0, c->stream>>>(c->d_lattice, (uint64_t)c->L * c->L / 32, replica,
                                                                       c->L, c->L / 32, x0 % c->L, y0 % c->L, w, h, d, d + n);
    cudaError_t e = cudaGetLastError();
    c->launches++;
    if (e == cudaSuccess) e = cudaMemcpyAsync(sx, d, n, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(sy, d + n, n, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    cudaFree(d);
    if (e != cudaSuccess) return fail(c, KPZ_ECUDA, "get_window: %s", cudaGetErrorString(e));
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
    if (replica >= c->R || !sx || !sy) return fail(c, KPZ_EINVAL, "bad argument");
    const size_t n = (size_t)c->L * c->L;
    int8_t* d = nullptr;
    if (cudaMalloc(&d, 2 * n) != cudaSuccess) { cudaGetLastError(); return fail(c, KPZ_ENOMEM, "temporary device buffer"); }
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
    if (e != cudaSuccess) return fail(c, KPZ_ECUDA, "set_slopes: %s", cudaGetErrorString(e));
    if (hflags & 1) return fail(c, KPZ_EINVAL, "slopes must be +1 or -1");
    if (hflags) return fail(c, KPZ_ESTATE, "state is not curl-free with zero tilt (flags %d)", hflags);
    return KPZ_OK;
}

int32_t kpz_state_hash(kpz_ctx* c, uint32_t replica, uint64_t* out) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if (replica >= c->R || !out) return fail(c, KPZ_EINVAL, "bad argument");
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
    if (replica >= c->R) return fail(c, KPZ_EINVAL, "replica out of range");
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
    if (!host_dst || bytes < c->lattice_bytes) return fail(c, KPZ_EINVAL, "host buffer too small");
    KPZ_CUDA(c, cudaMemcpyAsync(host_dst, c->d_lattice, c->lattice_bytes, cudaMemcpyDeviceToHost, c->stream));
    KPZ_CUDA(c, cudaStreamSynchronize(c->stream));
    return KPZ_OK;
}

int32_t kpz_import_packed(kpz_ctx* c, const void* host_src, size_t bytes, const int64_t* h00, uint64_t mcs) {
    int32_t rc = require_bound(c);
    if (rc != KPZ_OK) return rc;
    DeviceGuard dg__(c->device);
    if (!host_src || bytes < c->lattice_bytes || mcs > 0xFFFFFFFFull) return fail(c, KPZ_EINVAL, "bad argument");
    KPZ_CUDA(c, cudaMemcpyAsync(c->d_lattice, host_src, c->lattice_bytes, cudaMemcpyHostToDevice, c->stream));
    std::vector<unsigned long long> st((size_t)c->R * 4, 0ull);
    KPZ_CUDA(c, cudaMemcpyAsync(st.data(), c->d_scratch + c->sl.stats, (size_t)c->R * 32, cudaMemcpyDeviceToHost, c->stream));
    KPZ_CUDA(c, cudaStreamSynchronize(c->stream));
    for (uint32_t r = 0; r < c->R; ++r) { st[4 * r + 2] = (unsigned long long)(h00 ? h00[r] : 0); st[4 * r + 3] = 0ull; }
    KPZ_CUDA(c, cudaMemcpyAsync(c->d_scratch + c->sl.stats, st.data(), (size_t)c->R * 32, cudaMemcpyHostToDevice, c->stream));
    KPZ_CUDA(c, cudaStreamSynchronize(c->stream));
    c->mcs = mcs;
    c->attempts_base = mcs * (uint64_t)c->L * c->L;
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

// streams and events of one kpz_pipeline_host call, released on every return path
struct PipelineResources {
    cudaStream_t s_in = nullptr, s_out = nullptr;
    std::vector<cudaEvent_t> ev;
    ~PipelineResources() {
        for (cudaEvent_t e : ev) if (e) cudaEventDestroy(e);
        if (s_in) cudaStreamDestroy(s_in);
        if (s_out) cudaStreamDestroy(s_out);
    }
};

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
    if (!device_lattice2 || device_lattice2_bytes < c->lattice_bytes || ((uintptr_t)device_lattice2 & 15u))
        return fail(c, KPZ_EINVAL, "second device lattice missing, too small or not 16-byte aligned");
    if (n_lanes == 0 || n_rounds == 0 || !host_lattices || !mcs_start || bytes < c->lattice_bytes)
        return fail(c, KPZ_EINVAL, "bad argument");
    for (uint32_t l = 0; l < n_lanes; ++l) {
        if (!host_lattices[l]) return fail(c, KPZ_EINVAL, "NULL host lattice");
        if (mcs_start[l] + (uint64_t)n_rounds * mcs > 0xFFFFFFFFull) return fail(c, KPZ_EINVAL, "MCS clock would exceed 2^32-1");
    }
    const uint64_t B = (uint64_t)n_lanes * n_rounds;   // batches, b = round * n_lanes + lane
    PipelineResources res;
    KPZ_CUDA(c, cudaStreamCreateWithFlags(&res.s_in, cudaStreamNonBlocking));
    KPZ_CUDA(c, cudaStreamCreateWithFlags(&res.s_out, cudaStreamNonBlocking));
    res.ev.assign((size_t)B * 2, nullptr);               // per batch: copied in, copied out
    for (cudaEvent_t& e : res.ev) KPZ_CUDA(c, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    uint32_t* const dbuf[2] = {c->d_lattice, static_cast<uint32_t*>(device_lattice2)};
    std::vector<int64_t> h00((size_t)n_lanes * c->R, 0);
    if (h00_inout) std::memcpy(h00.data(), h00_inout, h00.size() * sizeof(int64_t));
    std::vector<uint64_t> clock(mcs_start, mcs_start + n_lanes);

    // host->device copy of batch b: its device slot must have been copied out (batch b-2), and so must the last
    // batch of the same lane (b - n_lanes), whose output is this batch's input
    auto enqueue_in = [&](uint64_t b) -> int32_t {
        if (b >= 2) KPZ_CUDA(c, cudaStreamWaitEvent(res.s_in, res.ev[2 * (b - 2) + 1], 0));
        if (b >= n_lanes) KPZ_CUDA(c, cudaStreamWaitEvent(res.s_in, res.ev[2 * (b - n_lanes) + 1], 0));
        KPZ_CUDA(c, cudaMemcpyAsync(dbuf[b & 1], host_lattices[b % n_lanes], c->lattice_bytes, cudaMemcpyHostToDevice, res.s_in));
        KPZ_CUDA(c, cudaEventRecord(res.ev[2 * b], res.s_in));
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
            KPZ_CUDA(c, cudaStreamWaitEvent(c->stream, res.ev[2 * b], 0));
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
            KPZ_CUDA(c, cudaEventRecord(res.ev[2 * b + 1], res.s_out));
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

// profiles of replica `replica` relative to h00 on the device (scratch prof[2][L]) + spectra; shared by the two calls
static int32_t run_profiles(kpz_ctx* c, uint32_t replica, bool with_fft, long long* h00_out) {
    const uint32_t L = c->L, W = L / 32;
    uint32_t logL = 0;
    while ((1u << logL) < L) ++logL;
    if (with_fft && (1u << logL) != L) return fail(c, KPZ_EINVAL, "the power spectrum needs L to be a power of two");
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
    if (replica >= c->R) return fail(c, KPZ_EINVAL, "replica out of range");
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
    if (replica >= c->R) return fail(c, KPZ_EINVAL, "replica out of range");
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

int32_t kpz_launch_count(const kpz_ctx* c, uint64_t* out) {
    if (!c || !out) return KPZ_EINVAL;
    *out = c->launches;
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
