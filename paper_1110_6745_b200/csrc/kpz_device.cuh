// kpz_device.cuh -- device code of the B200-native octahedron-KPZ hot path (sm_100a).
//
// Kernels:
//   kpz_update_kernel<T,...>   steps a2-a6 of SURVEY 8(a): tile + halo staged into shared memory as bit-lines,
//                              T*T sequential Philox-driven attempts per tile (eq. 2), write-back.
//   kpz_fill_flat_kernel       flat zig-zag start.
//   kpz_row0_prefix_kernel,    height reconstruction (eq. 3) as a per-column chunk monoid and the exact
//   kpz_column_chunk_kernel,   integer sums of h and h^2 (eq. 4).
//   kpz_combine_kernel
//   pack / unpack / hash / validation kernels for the parity and checkpoint calls of include/kpz.h.
//
// Nothing here is shared with oracle/ (own Philox, own rule, own height walk).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace kpz {

// ------------------------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  Ten rounds; the key schedule depends only on the seed, so
// the ten (k0,k1) pairs are formed from kernel parameters (uniform registers), not per call.
// ------------------------------------------------------------------------------------------------------------
#define KPZ_PHILOX_M0 0xD2511F53u
#define KPZ_PHILOX_M1 0xCD9E8D57u
#define KPZ_PHILOX_W0 0x9E3779B9u
#define KPZ_PHILOX_W1 0xBB67AE85u

struct PhiloxKey {
    uint32_t k0, k1;
};

__device__ __forceinline__ void philox_round(uint32_t& c0, uint32_t& c1, uint32_t& c2, uint32_t& c3, uint32_t k0,
                                             uint32_t k1) {
    const uint64_t p0 = (uint64_t)KPZ_PHILOX_M0 * c0;   // IMAD.WIDE.U32
    const uint64_t p1 = (uint64_t)KPZ_PHILOX_M1 * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;  // one LOP3
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    c1 = (uint32_t)p1;
    c3 = (uint32_t)p0;
    c0 = n0;
    c2 = n2;
}

__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, PhiloxKey key) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        philox_round(c0, c1, c2, c3, key.k0 + (uint32_t)r * KPZ_PHILOX_W0, key.k1 + (uint32_t)r * KPZ_PHILOX_W1);
    }
    return make_uint4(c0, c1, c2, c3);
}

__device__ __forceinline__ uint32_t mulhi32(uint32_t a, uint32_t n) { return __umulhi(a, n); }

// ------------------------------------------------------------------------------------------------------------
// Parameters shared by the update kernels.
// ------------------------------------------------------------------------------------------------------------
struct UpdateParams {
    uint32_t* lattice;             // device: packed lattice, all replicas
    unsigned long long* stats;     // device: [R][4] = deposits, removals, h00 (two's complement), reserved
    uint64_t plane_words;          // L*L/32
    uint64_t total_items;          // R * HN*HN  (tiles of one colour over all replicas)
    uint64_t thr_p, thr_q;         // accept iff (uint64)word < thr
    uint32_t L, NT, HN;            // lattice edge, tiles per edge, NT/2
    uint32_t W;                    // L/32: words per bit-line
    uint32_t tiles_per_colour;     // HN*HN
    uint32_t blocked;              // 1: 8x4 lane blocking of tiles (HN % 8 == 0), 0: linear
    uint32_t m;                    // MCS index (number of completed MCS)
    uint32_t slot;                 // 0..3: which entry of the colour order this launch executes
    PhiloxKey key;
};

// Global draw of MCS m for one replica: offset (multiples of 4 sites) and colour order.
// DESIGN.md "Schedule" S2.  Returns the colour processed in `slot`.
template <int T>
__device__ __forceinline__ void global_draw(const UpdateParams& P, uint32_t replica, uint32_t& ox, uint32_t& oy,
                                            uint32_t& colour) {
    const uint4 G = philox4x32_10(0u, 0xFFFFFFFFu, P.m, replica, P.key);
    constexpr uint32_t g = 4;
    ox = g * mulhi32(G.x, T / g);
    oy = g * mulhi32(G.y, T / g);
    const uint32_t pidx = mulhi32(G.z, 24u);
    // Lehmer decode of pidx into a permutation of {0,1,2,3}; pool kept as four 2-bit fields of one byte
    uint32_t pool = 0xE4u;   // fields (low to high): 0,1,2,3
    const uint32_t d[3] = {pidx / 6u, (pidx % 6u) / 2u, pidx % 2u};
    uint32_t perm[4];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        perm[k] = (pool >> (2u * d[k])) & 3u;
        const uint32_t low = pool & ((1u << (2u * d[k])) - 1u);
        pool = low | ((pool >> (2u * d[k] + 2u)) << (2u * d[k]));
    }
    perm[3] = pool & 3u;
    colour = P.slot == 0 ? perm[0] : P.slot == 1 ? perm[1] : P.slot == 2 ? perm[2] : perm[3];
}

// ------------------------------------------------------------------------------------------------------------
// Update kernel.  One THREAD owns one tile; the tile lives in shared memory as bit-lines:
//   plane X: line lx in [0,T] (a COLUMN of the tile; line T is the +x halo), bit ly  <=> sigma_x(X0+lx, Y0+ly)
//   plane Y: line ly in [0,T] (a ROW of the tile;    line T is the +y halo), bit lx  <=> sigma_y(X0+lx, Y0+ly)
// so that the pair (sigma_x(x,y), sigma_x(x+1,y)) is the same bit of two consecutive X lines and
// (sigma_y(x,y), sigma_y(x,y+1)) the same bit of two consecutive Y lines: no straddling, no halo special case.
// Word w of thread t sits at smem[w * NTHR + t]: every thread stays in its own bank -> conflict-free for any
// access pattern.  Threads never share data: no barrier anywhere in the kernel.
// ------------------------------------------------------------------------------------------------------------
template <int T>
struct TileGeom {
    static constexpr int LOG2T = (T == 4) ? 2 : (T == 8) ? 3 : (T == 16) ? 4 : (T == 32) ? 5 : 6;
    static constexpr int WPL = (T + 31) / 32;          // words per line
    static constexpr int LINES = T + 1;
    static constexpr int PLANE = LINES * WPL;
    static constexpr int WORDS = 2 * PLANE;            // per tile
    static constexpr uint32_t LINE_MASK = (T >= 32) ? 0xFFFFFFFFu : ((1u << (T & 31)) - 1u);
};

// loads T bits of a global bit-line starting at bit offset `o` (periodic in the line of W words)
template <int T, int NTHR>
__device__ __forceinline__ void load_line(const uint32_t* __restrict__ line, uint32_t W, uint32_t o, uint32_t* sm_line) {
    using G = TileGeom<T>;
    const uint32_t s = o & 31u;
    uint32_t a = o >> 5;
    uint32_t lo = __ldg(line + a);
#pragma unroll
    for (int k = 0; k < G::WPL; ++k) {
        uint32_t a1 = a + 1u;
        if (a1 == W) a1 = 0u;
        const uint32_t hi = __ldg(line + a1);
        uint32_t v = __funnelshift_r(lo, hi, s);
        if (T < 32) v &= G::LINE_MASK;
        sm_line[k * NTHR] = v;
        lo = hi;
        a = a1;
    }
}

// stores T bits back (read-modify-write of the partially covered edge words / bytes; see DESIGN.md
// "Halo write-back without races": no other active tile touches the same word (T >= 32) or byte (T < 32)).
template <int T, int NTHR>
__device__ __forceinline__ void store_line(uint32_t* __restrict__ line, uint32_t W, uint32_t o, const uint32_t* sm_line) {
    using G = TileGeom<T>;
    if (T >= 32) {
        const uint32_t s = o & 31u;
        uint32_t a = o >> 5;
        if (s == 0u) {
#pragma unroll
            for (int k = 0; k < G::WPL; ++k) {
                line[a] = sm_line[k * NTHR];
                a = (a + 1u == W) ? 0u : a + 1u;
            }
        } else {
            const uint32_t lowmask = (1u << s) - 1u;
            uint32_t prev = line[a] & lowmask;     // bits below the segment stay
            uint32_t carry = 0u;
#pragma unroll
            for (int k = 0; k < G::WPL; ++k) {
                const uint32_t v = sm_line[k * NTHR];
                const uint32_t out = (k == 0 ? prev : carry) | (v << s);
                line[a] = out;
                carry = v >> (32u - s);
                a = (a + 1u == W) ? 0u : a + 1u;
            }
            line[a] = (line[a] & ~lowmask) | carry;
        }
    } else {
        // byte granularity; o is a multiple of 4, T in {4, 8, 16}
        uint8_t* bl = reinterpret_cast<uint8_t*>(line);
        const uint32_t nbytes_line = W * 4u;
        const uint32_t v = sm_line[0] & G::LINE_MASK;
        const uint32_t sh = o & 7u;                          // 0 or 4
        const uint32_t span = v << sh;                       // <= 20 bits
        const uint32_t mask = G::LINE_MASK << sh;
        uint32_t b = o >> 3;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const uint32_t mk = (mask >> (8 * k)) & 0xFFu;
            if (mk) {
                const uint32_t nv = (span >> (8 * k)) & 0xFFu;
                if (mk == 0xFFu) bl[b] = (uint8_t)nv;
                else bl[b] = (uint8_t)((bl[b] & ~mk) | nv);
            }
            b = (b + 1u == nbytes_line) ? 0u : b + 1u;
        }
    }
}

// Stages / writes back one plane of a tile: lines line0 .. line0+T (periodic in L) of `plane`, T bits of each
// starting at bit offset o.  Global accesses are issued KPZ-batch lines at a time, all loads of a batch before the
// first dependent use, so that one thread keeps tens of requests in flight (one warp per CTA, ~6 warps per SM:
// memory-level parallelism has to come from inside the thread).
template <int T>
struct StageBatch {
    static constexpr int N = (T == 64) ? 13 : (T == 32) ? 11 : (T == 16) ? 17 : (T + 1);   // divides T+1
};

template <int T, int NTHR>
__device__ __forceinline__ void load_plane(const uint32_t* __restrict__ plane, uint32_t L, uint32_t W, uint32_t line0,
                                           uint32_t o, uint32_t* sm_plane) {
    using G = TileGeom<T>;
    constexpr int NB = StageBatch<T>::N;
    const uint32_t s = o & 31u;
    uint32_t idx[G::WPL + 1];
    idx[0] = o >> 5;
#pragma unroll
    for (int k = 1; k <= G::WPL; ++k) idx[k] = (idx[k - 1] + 1u == W) ? 0u : idx[k - 1] + 1u;
#pragma unroll 1
    for (int l0 = 0; l0 <= T; l0 += NB) {
        uint32_t raw[NB][G::WPL + 1];
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            uint32_t g = line0 + (uint32_t)(l0 + b);
            if (g >= L) g -= L;
            const uint32_t* line = plane + (size_t)g * W;
#pragma unroll
            for (int k = 0; k <= G::WPL; ++k) raw[b][k] = line[idx[k]];
        }
#pragma unroll
        for (int b = 0; b < NB; ++b) {
#pragma unroll
            for (int k = 0; k < G::WPL; ++k) {
                uint32_t v = __funnelshift_r(raw[b][k], raw[b][k + 1], s);
                if (T < 32) v &= G::LINE_MASK;
                sm_plane[((l0 + b) * G::WPL + k) * NTHR] = v;
            }
        }
    }
}

template <int T, int NTHR>
__device__ __forceinline__ void store_plane(uint32_t* __restrict__ plane, uint32_t L, uint32_t W, uint32_t line0,
                                            uint32_t o, const uint32_t* sm_plane) {
    using G = TileGeom<T>;
    if (T >= 32) {
        constexpr int NB = StageBatch<T>::N;
        const uint32_t s = o & 31u;
        uint32_t idx[G::WPL + 1];
        idx[0] = o >> 5;
#pragma unroll
        for (int k = 1; k <= G::WPL; ++k) idx[k] = (idx[k - 1] + 1u == W) ? 0u : idx[k - 1] + 1u;
        if (s == 0u) {
#pragma unroll 1
            for (int l0 = 0; l0 <= T; l0 += NB) {
#pragma unroll
                for (int b = 0; b < NB; ++b) {
                    uint32_t g = line0 + (uint32_t)(l0 + b);
                    if (g >= L) g -= L;
                    uint32_t* line = plane + (size_t)g * W;
#pragma unroll
                    for (int k = 0; k < G::WPL; ++k) line[idx[k]] = sm_plane[((l0 + b) * G::WPL + k) * NTHR];
                }
            }
        } else {
            // the first and last word of a line are shared with the (inactive) neighbour tiles: their bits are
            // re-read and merged.  No other active tile touches these words.
            const uint32_t lowmask = (1u << s) - 1u;
#pragma unroll 1
            for (int l0 = 0; l0 <= T; l0 += NB) {
                uint32_t first[NB], last[NB];
#pragma unroll
                for (int b = 0; b < NB; ++b) {
                    uint32_t g = line0 + (uint32_t)(l0 + b);
                    if (g >= L) g -= L;
                    const uint32_t* line = plane + (size_t)g * W;
                    first[b] = line[idx[0]];
                    last[b] = line[idx[G::WPL]];
                }
#pragma unroll
                for (int b = 0; b < NB; ++b) {
                    uint32_t g = line0 + (uint32_t)(l0 + b);
                    if (g >= L) g -= L;
                    uint32_t* line = plane + (size_t)g * W;
                    uint32_t carry = first[b] & lowmask;
#pragma unroll
                    for (int k = 0; k < G::WPL; ++k) {
                        const uint32_t v = sm_plane[((l0 + b) * G::WPL + k) * NTHR];
                        line[idx[k]] = carry | (v << s);
                        carry = v >> (32u - s);
                    }
                    line[idx[G::WPL]] = (last[b] & ~lowmask) | carry;
                }
            }
        }
    } else {
#pragma unroll 4
        for (int l = 0; l <= T; ++l) {
            uint32_t g = line0 + (uint32_t)l;
            if (g >= L) g -= L;
            store_line<T, NTHR>(plane + (size_t)g * W, W, o, sm_plane + (l * G::WPL) * NTHR);
        }
    }
}

// One attempt (eq. 2).  MODE 0: p = 1, q = 0 (accept word never needed -- bit-identical, the generator is
// counter-based).  MODE 1: general p, q.  TRACK: this thread's tile holds global site (0,0) at local index origin_idx.
// A flip is four shared-memory XOR reductions (ATOMS.XOR without return): no ALU work for the new words, and
// later loads of the same thread to the same address observe them (same-thread program order).
// Deposits are not counted here: n_dep - n_rem is recovered from the first moment of the X lines (weight_x below).
template <int T, int NTHR, int MODE, bool TRACK>
__device__ __forceinline__ void attempt(uint32_t* __restrict__ sm, uint32_t site_word, uint32_t accept_word,
                                        const UpdateParams& P, uint32_t& n_rem, int32_t& dh00, uint32_t origin_idx) {
    using G = TileGeom<T>;
    const uint32_t idx = site_word >> (32 - 2 * G::LOG2T);      // mulhi32(site_word, T*T)
    const uint32_t lx = idx & (uint32_t)(T - 1);
    const uint32_t ly = idx >> G::LOG2T;
    uint32_t* px = sm + (lx * G::WPL + (T > 32 ? (ly >> 5) : 0u)) * NTHR;
    uint32_t* py = sm + (G::PLANE + ly * G::WPL + (T > 32 ? (lx >> 5) : 0u)) * NTHR;
    const uint32_t xa = px[0], xb = px[G::WPL * NTHR];
    const uint32_t ya = py[0], yb = py[G::WPL * NTHR];
    const uint32_t bx = 1u << (ly & 31u);
    const uint32_t by = 1u << (lx & 31u);
    // local minimum: sigma_x(x)=-1, sigma_x(x+1)=+1, sigma_y(y)=-1, sigma_y(y+1)=+1  (bits 0,1,0,1)
    const bool is_min = ((~xa & xb & bx) != 0u) && ((~ya & yb & by) != 0u);
    bool flip;
    if (MODE == 0) {
        flip = is_min;
        if (TRACK) dh00 += (flip && idx == origin_idx) ? 2 : 0;
    } else {
        const bool is_max = ((xa & ~xb & bx) != 0u) && ((ya & ~yb & by) != 0u);
        const bool dep = is_min && ((uint64_t)accept_word < P.thr_p);
        const bool rem = is_max && ((uint64_t)accept_word < P.thr_q);
        flip = dep || rem;
        n_rem += rem ? 1u : 0u;
        if (TRACK) dh00 += (idx == origin_idx) ? (dep ? 2 : (rem ? -2 : 0)) : 0;
    }
    // unconditional XOR reductions with a zero mask when nothing flips: no branch, so the whole batch stays one
    // basic block for the instruction scheduler (ptxas branches around predicated ATOMS)
    const uint32_t mx = flip ? bx : 0u, my = flip ? by : 0u;
    atomicXor(px, mx);
    atomicXor(px + G::WPL * NTHR, mx);
    atomicXor(py, my);
    atomicXor(py + G::WPL * NTHR, my);
}

// T*T sequential attempts of one tile.  Philox calls are generated KPZ_BATCH at a time, one batch ahead of the
// attempts that consume them (the generator is counter-based, so the next batch does not depend on the lattice):
// the integer pipes work on batch b+1 while the shared-memory round trips of batch b are in flight.
template <int T, int NTHR, int MODE, bool TRACK>
__device__ __forceinline__ void run_tile_steps(uint32_t* __restrict__ sm, const UpdateParams& P, uint32_t tile_id,
                                               uint32_t replica, uint32_t& n_rem, int32_t& dh00,
                                               uint32_t origin_idx) {
    constexpr uint32_t CALLS = (uint32_t)(T * T) / 2u;
    constexpr uint32_t B = (CALLS >= 4u) ? 4u : CALLS;
    uint4 cur[B], nxt[B];
#pragma unroll
    for (uint32_t k = 0; k < B; ++k) cur[k] = philox4x32_10(k, tile_id, P.m, replica, P.key);
#pragma unroll 1
    for (uint32_t c = 0; c < CALLS; c += B) {
        // batch b+1 (the last iteration generates one unused batch: CALLS/B + 1 batches for CALLS/B used)
#pragma unroll
        for (uint32_t k = 0; k < B; ++k) nxt[k] = philox4x32_10(c + B + k, tile_id, P.m, replica, P.key);
#pragma unroll
        for (uint32_t k = 0; k < B; ++k) {
            attempt<T, NTHR, MODE, TRACK>(sm, cur[k].x, cur[k].y, P, n_rem, dh00, origin_idx);
            attempt<T, NTHR, MODE, TRACK>(sm, cur[k].z, cur[k].w, P, n_rem, dh00, origin_idx);
        }
#pragma unroll
        for (uint32_t k = 0; k < B; ++k) cur[k] = nxt[k];
    }
}

// first moment of the X lines of this thread's tile: sum over lines lx = 0..T of lx * popcount(line lx).
// A deposition at (lx,ly) moves a set bit from line lx+1 to line lx (-1), a removal does the opposite (+1):
// n_dep - n_rem = weight_before - weight_after.
template <int T, int NTHR>
__device__ __forceinline__ uint32_t weight_x(const uint32_t* __restrict__ sm) {
    using G = TileGeom<T>;
    uint32_t s = 0;
#pragma unroll 5
    for (int l = 1; l <= T; ++l) {
        uint32_t c = 0;
#pragma unroll
        for (int k = 0; k < G::WPL; ++k) c += __popc(sm[(l * G::WPL + k) * NTHR]);
        s += (uint32_t)l * c;
    }
    return s;
}

template <int T, int NTHR, int MODE>
__global__ void __launch_bounds__(NTHR) kpz_update_kernel(const UpdateParams P) {
    using G = TileGeom<T>;
    extern __shared__ uint32_t smem[];
    uint32_t* sm = smem + threadIdx.x;

    const uint64_t item = (uint64_t)blockIdx.x * NTHR + threadIdx.x;
    const bool active = item < P.total_items;
    uint32_t replica = 0, i = 0, j = 0;
    if (active) {
        replica = (uint32_t)(item / P.tiles_per_colour);
        const uint32_t wl = (uint32_t)(item - (uint64_t)replica * P.tiles_per_colour);
        if (P.blocked) {
            const uint32_t wq = wl >> 5, lane = wl & 31u;
            const uint32_t bpr = P.HN >> 3;
            const uint32_t bj = wq / bpr, bi = wq - bj * bpr;
            i = bi * 8u + (lane & 7u);
            j = bj * 4u + (lane >> 3);
        } else {
            j = wl / P.HN;
            i = wl - j * P.HN;
        }
    }
    uint32_t ox, oy, colour;
    global_draw<T>(P, replica, ox, oy, colour);
    const uint32_t tx = 2u * i + (colour & 1u), ty = 2u * j + (colour >> 1);
    const uint32_t X0 = ox + tx * T, Y0 = oy + ty * T;        // < L + T
    const uint32_t tile_id = ty * P.NT + tx;
    uint32_t* planeX = P.lattice + (size_t)replica * 2u * P.plane_words;
    uint32_t* planeY = planeX + P.plane_words;
    const uint32_t L = P.L, W = P.W;
    const uint32_t offX = (Y0 >= L) ? Y0 - L : Y0;   // bit offset inside an X line (a column): y direction
    const uint32_t offY = (X0 >= L) ? X0 - L : X0;   // bit offset inside a Y line (a row): x direction

    uint32_t n_dep = 0, n_rem = 0, w_before = 0;
    int32_t dh00 = 0;
    uint32_t origin_idx = 0xFFFFFFFFu;
    if (active) {
        // ---- a2: stage tile + halo ----
        load_plane<T, NTHR>(planeX, L, W, offY, offX, sm);
        load_plane<T, NTHR>(planeY, L, W, offX, offY, sm + G::PLANE * NTHR);
        // does this tile hold global site (0,0)?  local coordinates of it: (L - offY) mod L, (L - offX) mod L
        const uint32_t lx0 = (offY == 0u) ? 0u : L - offY;
        const uint32_t ly0 = (offX == 0u) ? 0u : L - offX;
        if (lx0 < (uint32_t)T && ly0 < (uint32_t)T) origin_idx = ly0 * T + lx0;
        w_before = weight_x<T, NTHR>(sm);
    }
    const bool any_origin = __any_sync(0xFFFFFFFFu, origin_idx != 0xFFFFFFFFu);
    if (active) {
        // ---- a3 + a4: T*T sequential attempts ----
        if (any_origin)
            run_tile_steps<T, NTHR, MODE, true>(sm, P, tile_id, replica, n_rem, dh00, origin_idx);
        else
            run_tile_steps<T, NTHR, MODE, false>(sm, P, tile_id, replica, n_rem, dh00, origin_idx);
        n_dep = w_before - weight_x<T, NTHR>(sm) + n_rem;
        // ---- a5: write back ----
        store_plane<T, NTHR>(planeX, L, W, offY, offX, sm);
        store_plane<T, NTHR>(planeY, L, W, offX, offY, sm + G::PLANE * NTHR);
    }
    // ---- a6: bookkeeping ----
    const uint32_t rep0 = __shfl_sync(0xFFFFFFFFu, replica, 0);
    const bool uniform = __all_sync(0xFFFFFFFFu, replica == rep0 && active);
    if (uniform) {
        uint32_t d = n_dep, r = n_rem;
        int32_t h = dh00;
#pragma unroll
        for (int sft = 16; sft > 0; sft >>= 1) {
            d += __shfl_xor_sync(0xFFFFFFFFu, d, sft);
            r += __shfl_xor_sync(0xFFFFFFFFu, r, sft);
            h += __shfl_xor_sync(0xFFFFFFFFu, h, sft);
        }
        if ((threadIdx.x & 31u) == 0u) {
            unsigned long long* st = P.stats + (size_t)rep0 * 4u;
            if (d) atomicAdd(st + 0, (unsigned long long)d);
            if (r) atomicAdd(st + 1, (unsigned long long)r);
            if (h) atomicAdd(st + 2, (unsigned long long)(long long)h);
        }
    } else if (active) {
        unsigned long long* st = P.stats + (size_t)replica * 4u;
        if (n_dep) atomicAdd(st + 0, (unsigned long long)n_dep);
        if (n_rem) atomicAdd(st + 1, (unsigned long long)n_rem);
        if (dh00) atomicAdd(st + 2, (unsigned long long)(long long)dh00);
    }
}

// ------------------------------------------------------------------------------------------------------------
// Flat start: sigma_x = sigma_y = +1 iff (x+y) odd.  One thread per 32-bit word of a replica's two planes.
// ------------------------------------------------------------------------------------------------------------
__global__ void kpz_fill_flat_kernel(uint32_t* lattice, uint64_t n_words_total, uint32_t W) {
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t w = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; w < n_words_total; w += stride) {
        // word w of a plane belongs to line (w / W); bit b of it is coordinate 32*(w % W) + b along the line.
        // (x+y) odd <=> (line + b) odd since 32*(w%W) is even: even line -> odd bits set.
        const uint64_t line = w / W;     // planes and replicas have L*W words each, L even: parity of line is global
        lattice[w] = (line & 1ull) ? 0x55555555u : 0xAAAAAAAAu;
    }
}

// ------------------------------------------------------------------------------------------------------------
// Measurement (eq. 3-4).  rel(x,y) = h(x,y) - h(0,0) = base(x) + l(x,y),
//   base(x) = sum_{l=1..x} sigma_x(l,0),   l(x,y) = sum_{k=1..y} sigma_y(x,k).
// Columns are cut into row chunks; a chunk with unknown entry height B contributes
//   sum (B+l) = n*B + S1,  sum (B+l)^2 = n*B^2 + 2*B*S1 + S2   with (S0 = exit l, S1 = sum l, S2 = sum l^2),
// so one pass over plane Y + a tiny combine gives the exact sums.
// ------------------------------------------------------------------------------------------------------------
__global__ void kpz_row0_prefix_kernel(const uint32_t* __restrict__ lattice, uint64_t plane_words, uint32_t L,
                                       uint32_t W, int32_t* __restrict__ base) {
    // one block per replica; thread t owns x in [t*seg, (t+1)*seg)
    __shared__ int32_t part[1024];
    const uint32_t replica = blockIdx.x;
    const uint32_t* planeX = lattice + (size_t)replica * 2u * plane_words;
    const uint32_t nthr = blockDim.x;
    const uint32_t seg = (L + nthr - 1u) / nthr;
    const uint32_t x0 = threadIdx.x * seg;
    int32_t s = 0;
    for (uint32_t x = x0; x < x0 + seg && x < L; ++x) {
        if (x > 0u) s += (int32_t)((planeX[(size_t)x * W] & 1u) << 1) - 1;    // sigma_x(x, 0)
    }
    part[threadIdx.x] = s;
    __syncthreads();
    // exclusive scan of the per-thread sums (Hillis-Steele on <= 1024 entries)
    for (uint32_t d = 1; d < nthr; d <<= 1) {
        int32_t v = (threadIdx.x >= d) ? part[threadIdx.x - d] : 0;
        __syncthreads();
        part[threadIdx.x] += v;
        __syncthreads();
    }
    int32_t run = part[threadIdx.x] - s;      // sum over x < x0
    int32_t* out = base + (size_t)replica * L;
    for (uint32_t x = x0; x < x0 + seg && x < L; ++x) {
        if (x > 0u) run += (int32_t)((planeX[(size_t)x * W] & 1u) << 1) - 1;
        out[x] = run;                         // h(x,0) - h(0,0)
    }
}

// grid (ceil(W/8), n_chunks, R), block 256: warp w of the block owns word-column 8*blockIdx.x + w, lane = bit.
__global__ void __launch_bounds__(256) kpz_column_chunk_kernel(const uint32_t* __restrict__ lattice,
                                                               uint64_t plane_words, uint32_t L, uint32_t W,
                                                               uint32_t rows_per_chunk, int32_t* __restrict__ cS0,
                                                               long long* __restrict__ cS1,
                                                               long long* __restrict__ cS2) {
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t wcol = blockIdx.x * 8u + (threadIdx.x >> 5);
    if (wcol >= W) return;
    const uint32_t chunk = blockIdx.y, replica = blockIdx.z, n_chunks = gridDim.y;
    const uint32_t* planeY = lattice + (size_t)replica * 2u * plane_words + plane_words;
    const uint32_t y_begin = chunk * rows_per_chunk;
    const uint32_t y_end = min(L, y_begin + rows_per_chunk);
    int32_t l = 0;
    long long s1 = 0, s2 = 0;
    for (uint32_t yb = y_begin; yb < y_end; yb += 32u) {
        // lane k fetches the word of row yb+k; rows are then consumed in order via shuffles
        const uint32_t yr = yb + lane;
        const uint32_t mine = (yr < y_end) ? __ldg(planeY + (size_t)yr * W + wcol) : 0u;
        const uint32_t nrow = min(32u, y_end - yb);
        int32_t t1 = 0;
        for (uint32_t k = 0; k < nrow; ++k) {
            const uint32_t word = __shfl_sync(0xFFFFFFFFu, mine, (int)k);
            const int32_t sig = (int32_t)(((word >> lane) & 1u) << 1) - 1;
            if (yb + k > 0u) l += sig;                       // row 0 carries no sigma_y step (eq. 3)
            t1 += l;
            s2 += (long long)l * (long long)l;
        }
        s1 += t1;
    }
    const size_t o = ((size_t)replica * n_chunks + chunk) * L + (size_t)wcol * 32u + lane;
    cS0[o] = l;
    cS1[o] = s1;
    cS2[o] = s2;
}

// grid (ceil(L/256), R), block 256: one thread per column; out[replica][4] += {lo(S1), hi(S1), lo(S2), hi(S2)}
__global__ void __launch_bounds__(256) kpz_combine_kernel(const int32_t* __restrict__ base,
                                                          const int32_t* __restrict__ cS0,
                                                          const long long* __restrict__ cS1,
                                                          const long long* __restrict__ cS2, uint32_t L,
                                                          uint32_t n_chunks, uint32_t rows_per_chunk,
                                                          unsigned long long* __restrict__ msum) {
    const uint32_t replica = blockIdx.y;
    const uint32_t x = blockIdx.x * 256u + threadIdx.x;
    long long a1 = 0, a2 = 0;
    if (x < L) {
        long long B = base[(size_t)replica * L + x];
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t y_begin = c * rows_per_chunk;
            if (y_begin >= L) break;
            const long long n = (long long)(min(L, y_begin + rows_per_chunk) - y_begin);
            const size_t o = ((size_t)replica * n_chunks + c) * L + x;
            const long long S1 = cS1[o], S2 = cS2[o];
            a1 += n * B + S1;
            a2 += n * B * B + 2 * B * S1 + S2;
            B += cS0[o];
        }
    }
    // split into 32-bit halves so that the cross-column sums cannot overflow 64 bits; warp + block reduce
    unsigned long long v[4] = {(unsigned long long)(uint32_t)a1, (unsigned long long)(a1 >> 32),
                               (unsigned long long)(uint32_t)a2, (unsigned long long)(a2 >> 32)};
    __shared__ unsigned long long red[8][4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
#pragma unroll
        for (int sft = 16; sft > 0; sft >>= 1) v[q] += __shfl_xor_sync(0xFFFFFFFFu, v[q], sft);
    }
    if ((threadIdx.x & 31u) == 0u) {
#pragma unroll
        for (int q = 0; q < 4; ++q) red[threadIdx.x >> 5][q] = v[q];
    }
    __syncthreads();
    if (threadIdx.x < 4u) {
        unsigned long long t = 0;
        for (int w = 0; w < 8; ++w) t += red[w][threadIdx.x];
        atomicAdd(msum + (size_t)replica * 4u + threadIdx.x, t);
    }
}

// ------------------------------------------------------------------------------------------------------------
// Parity / checkpoint helpers.
// ------------------------------------------------------------------------------------------------------------
// window unpack: out arrays [j*w + i] <- sigma(x0+i, y0+j), periodic
__global__ void kpz_unpack_window_kernel(const uint32_t* __restrict__ lattice, uint64_t plane_words, uint32_t replica,
                                         uint32_t L, uint32_t W, uint32_t x0, uint32_t y0, uint32_t w, uint32_t h,
                                         int8_t* __restrict__ sx, int8_t* __restrict__ sy) {
    const uint32_t* planeX = lattice + (size_t)replica * 2u * plane_words;
    const uint32_t* planeY = planeX + plane_words;
    const uint64_t n = (uint64_t)w * h;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += stride) {
        const uint32_t jj = (uint32_t)(t / w), ii = (uint32_t)(t - (uint64_t)jj * w);
        const uint32_t x = (x0 + ii) % L, y = (y0 + jj) % L;
        const uint32_t bxv = (planeX[(size_t)x * W + (y >> 5)] >> (y & 31u)) & 1u;
        const uint32_t byv = (planeY[(size_t)y * W + (x >> 5)] >> (x & 31u)) & 1u;
        sx[t] = bxv ? 1 : -1;
        sy[t] = byv ? 1 : -1;
    }
}

// validation of host slopes already copied to the device: flags[0] |= 1 (value not +-1), |= 2 (curl), |= 4 (tilt)
__global__ void kpz_validate_kernel(const int8_t* __restrict__ sx, const int8_t* __restrict__ sy, uint32_t L,
                                    int* __restrict__ flags) {
    const uint64_t n = (uint64_t)L * L;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    int bad = 0;
    for (uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; t < n; t += stride) {
        const uint32_t y = (uint32_t)(t / L), x = (uint32_t)(t - (uint64_t)y * L);
        const int a = sx[t], b = sy[t];
        if ((a != 1 && a != -1) || (b != 1 && b != -1)) bad |= 1;
        const uint32_t x1 = (x + 1u == L) ? 0u : x + 1u, y1 = (y + 1u == L) ? 0u : y + 1u;
        const int lhs = sx[(size_t)y * L + x1] + sy[(size_t)y1 * L + x1];
        const int rhs = sy[(size_t)y1 * L + x] + sx[(size_t)y1 * L + x1];
        if (lhs != rhs) bad |= 2;
    }
    // tilt: thread t < L checks row t of sx and column t of sy
    for (uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; t < L; t += stride) {
        int rs = 0, cs = 0;
        for (uint32_t k = 0; k < L; ++k) {
            rs += sx[(size_t)t * L + k];
            cs += sy[(size_t)k * L + t];
        }
        if (rs != 0 || cs != 0) bad |= 4;
    }
    if (bad) atomicOr(flags, bad);
}

// pack: one thread per word of plane X and of plane Y
__global__ void kpz_pack_kernel(uint32_t* __restrict__ lattice, uint64_t plane_words, uint32_t replica, uint32_t L,
                                uint32_t W, const int8_t* __restrict__ sx, const int8_t* __restrict__ sy) {
    uint32_t* planeX = lattice + (size_t)replica * 2u * plane_words;
    uint32_t* planeY = planeX + plane_words;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; t < plane_words; t += stride) {
        const uint32_t line = (uint32_t)(t / W), k = (uint32_t)(t - (uint64_t)line * W);
        uint32_t wx = 0, wy = 0;
        for (uint32_t b = 0; b < 32u; ++b) {
            const uint32_t c = 32u * k + b;
            // plane X: line = x, c = y ; plane Y: line = y, c = x
            if (sx[(size_t)c * L + line] > 0) wx |= 1u << b;
            if (sy[(size_t)line * L + c] > 0) wy |= 1u << b;
        }
        planeX[t] = wx;
        planeY[t] = wy;
    }
}

__device__ __forceinline__ uint64_t mix64(uint64_t z) {
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

// state hash: one thread per 32-bit word of plane Y (row y, columns 32k..32k+31) and the matching X bits
__global__ void kpz_hash_kernel(const uint32_t* __restrict__ lattice, uint64_t plane_words, uint32_t replica,
                                uint32_t L, uint32_t W, unsigned long long* __restrict__ out) {
    const uint32_t* planeX = lattice + (size_t)replica * 2u * plane_words;
    const uint32_t* planeY = planeX + plane_words;
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    unsigned long long acc = 0;
    for (uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; t < plane_words; t += stride) {
        const uint32_t line = (uint32_t)(t / W), k = (uint32_t)(t - (uint64_t)line * W);
        const uint32_t wy = planeY[t];      // row y = line, x = 32k + b
        const uint32_t wx = planeX[t];      // column x = line, y = 32k + b
        for (uint32_t b = 0; b < 32u; ++b) {
            const uint32_t c = 32u * k + b;
            if ((wy >> b) & 1u) acc += mix64(2ull * ((uint64_t)line * L + c) + 1ull);
            if ((wx >> b) & 1u) acc += mix64(2ull * ((uint64_t)c * L + line));
        }
    }
#pragma unroll
    for (int sft = 16; sft > 0; sft >>= 1) acc += __shfl_xor_sync(0xFFFFFFFFu, acc, sft);
    if ((threadIdx.x & 31u) == 0u && acc) atomicAdd(out, acc);
}

__global__ void kpz_philox_selftest_kernel(const uint32_t* ctr, const uint32_t* key, uint32_t* out, uint32_t n) {
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n) return;
    PhiloxKey k{key[2 * t], key[2 * t + 1]};
    const uint4 r = philox4x32_10(ctr[4 * t], ctr[4 * t + 1], ctr[4 * t + 2], ctr[4 * t + 3], k);
    out[4 * t] = r.x; out[4 * t + 1] = r.y; out[4 * t + 2] = r.z; out[4 * t + 3] = r.w;
}

}  // namespace kpz
