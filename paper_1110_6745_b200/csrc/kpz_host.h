// kpz_host.h -- internal host-side declarations shared by the translation units of libkpz_b200.so (not installed;
// the public interface is include/kpz.h).  The kernel instantiations are spread over several .cu files so that nvcc
// can compile them in parallel; each of those files exports one launcher declared here.
#pragma once
#include "../../include/kpz.h"

#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdio>
#include <vector>

#include "kpz_device.cuh"

#define KPZ_HIDDEN __attribute__((visibility("hidden")))

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
    uint32_t n_slabs, slab;  // > 0: this handle holds slab `slab` of n_slabs of one lattice (kpz_create_slab); 0: a whole lattice
    uint32_t rows_own, rows; // slab: rows of the lattice this slab owns, rows stored (owned + ghost rows of the next slab)
    int device;              // ordinal of the device that holds the bound buffers (-1 before kpz_bind)
    cudaStream_t s_in, s_out;     // copy streams of kpz_pipeline_host, created on first use, kept for the handle's life
    std::vector<cudaEvent_t> events;   // its event pool (grown on demand, destroyed with the handle)
    char err[512];
};

inline int32_t kpz_fail(kpz_ctx* c, int32_t code, const char* fmt, ...) {
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
            return kpz_fail((c), KPZ_ECUDA, "%s failed: %s", #expr, cudaGetErrorString(e__));      \
    } while (0)

constexpr int KPZ_MAX_DEVICES = 64;
constexpr size_t KPZ_RESIDENT_SMEM_MAX = 200 * 1024;

// launch shape of the lattice-resident kernel for one handle (kpz.cu: resident_plan)
struct ResidentPlan {
    bool ok;            // the lattices and the tiles fit in shared memory and the schedule is the default one
    uint32_t G, nthr, blocks;
    size_t smem;
};

// one launcher per translation unit (tile sizes 64 / 32 and 16 / 8 / 4)
KPZ_HIDDEN int32_t kpz_launch_update_wide(kpz_ctx* c, const kpz::UpdateParams& P);
KPZ_HIDDEN int32_t kpz_launch_update_narrow(kpz_ctx* c, const kpz::UpdateParams& P);
KPZ_HIDDEN int32_t kpz_launch_resident_wide(kpz_ctx* c, const kpz::UpdateParams& P, const ResidentPlan& pl, uint32_t n_mcs);
KPZ_HIDDEN int32_t kpz_launch_resident_narrow(kpz_ctx* c, const kpz::UpdateParams& P, const ResidentPlan& pl, uint32_t n_mcs);
