// kpz_peaks.cuh -- micro-benchmarks of the pipes that bound kpz_update_kernel.
//
// MEASURED_PEAKS.json carries HBM bandwidth and bf16 tensor throughput only; the update kernel is bound by the
// integer ALU pipe (LOP3 / SHF / LEA) and by the shared-memory data pipe (LDS / ATOMS wavefronts), so their peaks
// are measured here, on the box, by kernels that do nothing but issue one kind of instruction from every warp
// slot of every SM.  Each kernel runs ITER iterations of an unrolled body of independent chains (eight registers,
// so that neither latency nor the register file limits the issue rate); its rate is instructions x 32 lanes /
// CUDA-event time.  The SM clock during the measurement is read back as clock64() ticks / globaltimer nanoseconds of one thread.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "kpz_device.cuh"

namespace kpz {

enum PeakKind { PEAK_LOP3 = 0, PEAK_SHF = 1, PEAK_IMAD = 2, PEAK_IMAD_WIDE = 3, PEAK_LDS = 4, PEAK_ATOMS = 5, PEAK_MIX = 6 };

constexpr int PEAK_UNROLL = 64;      // instructions of the measured kind per loop iteration and chain group

template <int KIND>
__global__ void __launch_bounds__(256) kpz_peak_kernel(uint32_t iters, uint32_t seed, uint32_t* __restrict__ sink,
                                                       unsigned long long* __restrict__ ticks) {
    __shared__ uint32_t sm[32 * 64 + 256];
    uint32_t r[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) r[k] = seed * (2u * k + 1u) + threadIdx.x;
    for (uint32_t i = threadIdx.x; i < 32 * 64 + 256; i += blockDim.x) sm[i] = i * seed;
    __syncthreads();
    // word w of lane t at sm[w * 32 + lane]: every lane in its own bank, as in the update kernel
    uint32_t* mine = sm + (threadIdx.x & 31u);
    // SM clock = clock64 ticks per globaltimer nanosecond of the same thread (independent of how the scheduler
    // interleaves the CTAs of an SM)
    unsigned long long g0, g1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
    const long long t0 = clock64();
#pragma unroll 1
    for (uint32_t it = 0; it < iters; ++it) {
#pragma unroll
        for (int j = 0; j < PEAK_UNROLL / 8; ++j) {
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                if (KIND == PEAK_LOP3) {
                    asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(r[k]) : "r"(r[(k + 1) & 7]), "r"(seed));
                } else if (KIND == PEAK_SHF) {
                    asm volatile("shf.l.wrap.b32 %0, %0, %1, 7;" : "+r"(r[k]) : "r"(r[(k + 3) & 7]));
                } else if (KIND == PEAK_IMAD) {
                    asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(r[k]) : "r"(seed), "r"(r[(k + 1) & 7]));
                } else if (KIND == PEAK_IMAD_WIDE) {
                    unsigned long long w;
                    asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(w) : "r"(r[k]), "r"(0xD2511F53u));
                    r[k] = (uint32_t)(w >> 32) ^ (uint32_t)w;       // one LOP3 per multiply rides along (Philox does the same)
                } else if (KIND == PEAK_LDS) {
                    uint32_t v;
                    // ld.volatile: ptxas would hoist a plain load from a loop-invariant address out of the loop
                    asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(v) : "r"((uint32_t)__cvta_generic_to_shared(mine + 32 * ((j * 8 + k) & 63))) : "memory");
                    r[k] ^= v;
                } else if (KIND == PEAK_ATOMS) {
                    asm volatile("red.shared.xor.b32 [%0], %1;" ::"r"((uint32_t)__cvta_generic_to_shared(mine + 32 * ((j * 8 + k) & 63))), "r"(r[k]) : "memory");
                } else {
                    // the instruction mix of one p = 1 attempt: 5 LDS, 2 SHF, 3 LOP3, 1 ATOMS on private banks
                    uint32_t a, b, c, d, e;
                    const uint32_t base = (uint32_t)__cvta_generic_to_shared(mine + 32 * ((r[k] >> 27) + 2 * k));
                    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(a) : "r"(base));
                    asm volatile("ld.shared.u32 %0, [%1+128];" : "=r"(b) : "r"(base));
                    asm volatile("ld.shared.u32 %0, [%1+256];" : "=r"(c) : "r"(base));
                    asm volatile("ld.shared.u32 %0, [%1+384];" : "=r"(d) : "r"(base));
                    asm volatile("ld.shared.u32 %0, [%1+512];" : "=r"(e) : "r"(base));
                    const uint32_t wl = __funnelshift_l(a, b, 1), wr = __funnelshift_r(b, c, 1);
                    uint32_t t1, t2, md;
                    asm volatile("lop3.b32 %0, %1, %2, %3, 0xdb;" : "=r"(t1) : "r"(b), "r"(wl), "r"(wr));
                    asm volatile("lop3.b32 %0, %1, %2, %3, 0xbd;" : "=r"(t2) : "r"(b), "r"(d), "r"(e));
                    asm volatile("lop3.b32 %0, %1, %2, %3, 0x10;" : "=r"(md) : "r"(r[k]), "r"(t1), "r"(t2));
                    asm volatile("red.shared.xor.b32 [%0+128], %1;" ::"r"(base), "r"(md & 1u) : "memory");
                    r[k] = r[k] * 0x9E3779B9u + md;
                }
            }
        }
    }
    const long long t1 = clock64();
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
    uint32_t acc = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) acc ^= r[k];
    if (acc == 0x12345678u) sink[blockIdx.x] = acc + sm[threadIdx.x];      // keeps the chains alive, never true in practice
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        ticks[0] = (unsigned long long)(t1 - t0);
        ticks[1] = g1 - g0;
    }
}

// The dependent chain of one tile: 5 LDS (random row of a private 66-row tile) -> 2 funnel shifts -> 3 LOP3 -> XOR
// reduction, the next attempt's loads issued after the reduction as in the update kernel (the site sequence does not
// depend on the tile).  One CTA on one SM; reports clock64 ticks per attempt of warp 0 -- the latency that only other
// warps can hide.  With w warps per scheduler the per-scheduler cost follows 17 + 48 / w cycles on B200.
__global__ void __launch_bounds__(512) kpz_chain_kernel(uint32_t iters, uint32_t seed, unsigned long long* __restrict__ ticks) {
    __shared__ uint32_t sm[32 * 72];
    for (uint32_t i = threadIdx.x; i < 32 * 72; i += blockDim.x) sm[i] = i * 2654435761u ^ seed;
    __syncthreads();
    uint32_t* mine = sm + (threadIdx.x & 31u);
    uint32_t w = seed + threadIdx.x;
    const long long t0 = clock64();
#pragma unroll 4
    for (uint32_t it = 0; it < iters; ++it) {
        w = w * 1664525u + 1013904223u;
        uint32_t* a = mine + 32u * ((w >> 26) + 2u);
        const uint32_t wo = a[0], wd = a[-32], wu = a[32], wp = a[-64], wn = a[64];
        const uint32_t wl = __funnelshift_l(wp, wo, 1), wr = __funnelshift_r(wo, wn, 1);
        const uint32_t t1 = (wo ^ ~wl) | (wo ^ wr), t2 = (wo ^ wu) | (wo ^ ~wd);
        atomicXor(a, (1u << ((w >> 20) & 31u)) & ~t1 & ~t2);
    }
    const long long t1 = clock64();
    if (threadIdx.x == 0) ticks[0] = (unsigned long long)(t1 - t0);
}


// ---- the attempt loop alone, in two tile layouts (fewer words per tile) -------------------
// Shared memory decides the occupancy of the T = 64 kernel: 199 words per tile = 9 warps per SM.  LAYOUT 0 runs the
// update kernel's own attempt loop (run_tile_steps, MODE 0) on a tile of random bits without the staging -- the ceiling of
// the present layout.  LAYOUT 1 is the cheapest layout with fewer words that was found: the 66 x 66 bits of tile and halo as
// ONE bit string with a row pitch of 66 bits (138 words = 12 warps per SM).  Left / right neighbours then need no halo word
// (the funnel shifts cross the row ends by themselves), but the rows above and below sit 2 bits off and need a rotate
// each, and three word indices instead of one.  Same Philox calls, same five loads, tests and XOR reduction; what is
// measured is whether three more warps per SM pay for the two rotates and the address arithmetic.  NOT a kernel of the
// path: the tile holds random bits and nothing is written back.
constexpr int LAYOUT66_WORDS = 138;

template <int NTHR>
__device__ __forceinline__ void attempt_pitch66(uint32_t* __restrict__ sm, uint32_t site_word, float& dep_f, uint32_t two,
                                                uint32_t two27) {
    const uint32_t idx = site_word >> 20, ly = site_word >> 26;
    // q = ly * 66 + lx: bit position of the site in the string, + 96.  The multiplier pipe is the idle one: q by IMAD, the
    // word indices of the rows above / below as the high halves of q * 2^27 + c * 2^27 (IMAD.WIDE) instead of add + shift
    // (the multipliers 2 and 2^27 arrive as kernel arguments: ptxas turns constant powers of two back into shifts and adds)
    uint32_t q;
    asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(q) : "r"(ly), "r"(two), "r"(idx));
    unsigned long long pu, pd;
    asm("mad.wide.u32 %0, %1, %2, %3;" : "=l"(pu) : "r"(q), "r"(two27), "l"(162ull << 27));
    asm("mad.wide.u32 %0, %1, %2, %3;" : "=l"(pd) : "r"(q), "r"(two27), "l"(30ull << 27));
    uint32_t* a = sm + ((q >> 5) + 3u) * NTHR;
    const uint32_t wo = a[0], wp = *(a - NTHR), wn = a[NTHR];
    const uint32_t wu = sm[(uint32_t)(pu >> 32) * NTHR];    // bit (q + 2) & 31 of the word that holds position + 66
    const uint32_t wd = sm[(uint32_t)(pd >> 32) * NTHR];    // bit (q - 2) & 31 of the word that holds position - 66
    const uint32_t wl = __funnelshift_l(wp, wo, 1), wr = __funnelshift_r(wo, wn, 1);
    const uint32_t wua = __funnelshift_r(wu, wu, 2), wda = __funnelshift_l(wd, wd, 2);
    const uint32_t bit = __funnelshift_l(0u, 1u, q);
    const uint32_t t1 = lop3<0xDB>(wo, wl, wr), t2 = lop3<0xBD>(wo, wua, wda);
    const uint32_t md0 = lop3_and_not_not(bit, t1, t2);
    atomicXor(a, md0);
    asm("{ .reg .pred p; setp.ne.u32 p, %1, 0; @p add.f32 %0, %0, 0f3F800000; }" : "+f"(dep_f) : "r"(md0));
}

template <int LAYOUT>
__global__ void __launch_bounds__(96, LAYOUT ? 4 : 3) kpz_layout_kernel(uint32_t seed, uint32_t m, uint32_t two, uint32_t two27,
                                                                             uint32_t* __restrict__ sink) {
    constexpr int NTHR = 96;
    constexpr int WORDS = LAYOUT ? LAYOUT66_WORDS : TileGeom<64>::WORDS;
    extern __shared__ uint32_t smem[];
    uint32_t* sm = smem + threadIdx.x;
    const uint32_t tile_id = blockIdx.x * NTHR + threadIdx.x;
    for (int w = 0; w < WORDS; ++w) sm[w * NTHR] = (tile_id * 2654435761u + (uint32_t)w * 0x9E3779B9u) ^ seed;
    UpdateParams P = {};
    P.key.k0 = seed;
    P.key.k1 = ~seed;
    P.m = m;
    uint32_t n_dep = 0, n_rem = 0;
    int32_t dh00 = 0;
    if (LAYOUT == 0) {
        run_tile_steps<64, NTHR, 0, false, false, 0>(sm, P, tile_id, 0u, n_dep, n_rem, dh00, 0xFFFFFFFFu, 0u);
    } else {
        float dep_f = 0.0f;
        uint4 cur = philox4x32_10(0u, tile_id, P.m, 0u, P.key), nxt;
#pragma unroll 4
        for (uint32_t c = 0; c < 512u; ++c) {
            nxt = philox4x32_10(c + 1u, tile_id, P.m, 0u, P.key);
            attempt_pitch66<NTHR>(sm, cur.x, dep_f, two, two27);
            attempt_pitch66<NTHR>(sm, cur.x * 4096u, dep_f, two, two27);
            attempt_pitch66<NTHR>(sm, cur.y, dep_f, two, two27);
            attempt_pitch66<NTHR>(sm, cur.y * 4096u, dep_f, two, two27);
            attempt_pitch66<NTHR>(sm, cur.z, dep_f, two, two27);
            attempt_pitch66<NTHR>(sm, cur.z * 4096u, dep_f, two, two27);
            attempt_pitch66<NTHR>(sm, cur.w, dep_f, two, two27);
            attempt_pitch66<NTHR>(sm, cur.w * 4096u, dep_f, two, two27);
            cur = nxt;
        }
        n_dep = (uint32_t)dep_f;
    }
    uint32_t acc = n_dep;
    for (int w = 0; w < WORDS; ++w) acc ^= sm[w * NTHR];
    if (acc == 0x12345678u) sink[0] = acc;       // keeps the tile alive, practically never true
}

}  // namespace kpz
