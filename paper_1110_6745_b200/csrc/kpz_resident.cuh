// kpz_resident.cuh -- lattice-resident update kernels for small lattices (L a power of two, L*L/8 bytes of
// height bits per replica in shared memory): BASELINE configs 1, 2-shaped small cases and the L <= 512 ensembles of
// config 4.  Same schedule S1-S4, same Philox streams, bit-identical to kpz_update_kernel.
//
// What differs from the tiled kernel (kpz_device.cuh) is only WHERE the height bits live:
//   * one CTA loads the WHOLE lattice of its replica(s) once, converts slopes to one height bit per site
//     (u = h1 ^ E as in kpz_device.cuh, but in GLOBAL coordinates: the periodic lattice needs no halo at all),
//     runs n MCS -- the four colour passes of an MCS separated by __syncthreads() instead of kernel launches, the
//     global draw (S2) evaluated in-kernel -- and converts back once at the end.  No per-tile staging, no launch per
//     colour: the 4 x n launches of a kpz_run(n) become one.
//   * kpz_resident_kernel<.., COOP = false>: one THREAD per tile as in the tiled kernel (sequential order = program
//     order).  For ensembles with many tiles in flight (config 4: 1024 x L = 128).
//   * kpz_resident_kernel<.., COOP = true>: one WARP per tile, "warp-cooperative sequential updates": the 32 lanes
//     take 32 consecutive steps of the tile's stream at once.  A bitmap M of the local minima (and one of the maxima)
//     of the whole lattice is kept next to u; a lane whose site is not flippable is done after one load.  The
//     flippable lanes are served in step order: the lowest one flips (XOR of its bit in u), the words of M around
//     it are recomputed by five lanes, the later lanes re-read their bit of M (only sites within distance 1 of a
//     flip can change status, and M tracks exactly that), and so on.  Every step sees the state its predecessors
//     left, so the result is the sequential one; a tile's T*T dependent round trips become T*T/32 + (number of
//     flips).  For lattices with few tiles (config 1: 64 per colour), which are bound by one tile's chain.
//
// Same-colour tiles are processed concurrently by different threads / warps of the CTA.  They may share 32-bit
// words of u and M (tile origins are multiples of 4, not 32), so every update of a word is an atomic XOR of the
// bits the tile owns: its own sites in u; the sites within distance 1 of its own sites in M (two same-colour
// tiles are at least one tile apart, so these sets are disjoint).
#pragma once
#include "kpz_device.cuh"

namespace kpz {

struct ResidentParams {
    uint32_t* lattice;             // device: packed lattice, all replicas
    unsigned long long* stats;     // device: [R][4]
    uint64_t plane_words;          // L*L/32
    uint64_t thr_p, thr_q;         // accept iff (uint64)word < thr
    uint32_t L, W, NT, HN;         // lattice edge (power of two), L/32, tiles per edge, NT/2
    uint32_t tpc;                  // HN*HN tiles per colour and replica
    uint32_t R, G;                 // replicas in the handle, replicas per CTA
    uint32_t m0, n_mcs;            // MCS clock at entry, MCS to run
    PhiloxKey key;
};

// colour order of one MCS (S2) as four 2-bit fields, plus the origin
template <int T>
__device__ __forceinline__ void resident_draw(PhiloxKey key, uint32_t m, uint32_t replica, uint32_t& ox, uint32_t& oy,
                                              uint32_t& perm) {
    const uint4 G = philox4x32_10(0u, 0xFFFFFFFFu, m, replica, key);
    ox = 4u * mulhi32(G.x, T / 4);
    oy = 4u * mulhi32(G.y, T / 4);
    const uint32_t pidx = mulhi32(G.z, 24u);
    uint32_t pool = 0xE4u;
    const uint32_t d[3] = {pidx / 6u, (pidx % 6u) / 2u, pidx % 2u};
    perm = 0u;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        perm |= ((pool >> (2u * d[k])) & 3u) << (2 * k);
        const uint32_t low = pool & ((1u << (2u * d[k])) - 1u);
        pool = low | ((pool >> (2u * d[k] + 2u)) << (2u * d[k]));
    }
    perm |= (pool & 3u) << 6;
}

// the two neighbour tests of eq. 2 in the parity-free encoding (kpz_device.cuh, attempt<>), whole words:
// bit set <=> the site is a local minimum / maximum.  wp / wn: the words left / right of wo in the same row.
__device__ __forceinline__ void minmax_words(uint32_t wo, uint32_t wp, uint32_t wn, uint32_t wu, uint32_t wd,
                                             uint32_t& mn, uint32_t& mx) {
    const uint32_t wl = __funnelshift_l(wp, wo, 1), wr = __funnelshift_r(wo, wn, 1);
    mn = ~(lop3<0xDB>(wo, wl, wr) | lop3<0xBD>(wo, wu, wd));
    mx = ~(lop3<0xBD>(wo, wl, wr) | lop3<0xDB>(wo, wu, wd));
}

// ---- slopes (HBM) -> u (shared memory), whole periodic lattice of one replica ---------------------------------
// phase 1 (all threads of the group): raw sigma_y words into u;  phase 2 (one thread per word column): the
// recurrence h1(.,y) = h1(.,y-1) ^ sigma_y(.,y) ^ ycode(y) down the column, row 0 from the prefix XOR of sigma_x.
__device__ __forceinline__ void resident_load(const uint32_t* __restrict__ planeX, const uint32_t* __restrict__ planeY,
                                              uint32_t L, uint32_t W, uint32_t* __restrict__ u, uint32_t tid, uint32_t nthr) {
    const uint32_t n = L * W;
    for (uint32_t i = tid; i < n; i += nthr) u[i] = planeY[i];
    __syncthreads();
    for (uint32_t k = tid; k < W; k += nthr) {
        uint32_t carry = 0u, prev = 0u;
        for (uint32_t j = 0; j <= k; ++j) {
            uint32_t t = planeX[j] ^ 0xAAAAAAAAu;      // h1(x,0) = XOR_{l=1..x} XNOR(sigma_x(l,0), h0(l-1,0))
            if (j == 0u) t &= ~1u;                     // anchor h1(0,0) = 0
            t = prefix_xor32(t) ^ carry;
            carry = 0u - (t >> 31);
            prev = t;
        }
        u[k] = prev ^ enc_word(0u);
        for (uint32_t y = 1; y < L; ++y) {
            const uint32_t cur = prev ^ u[y * W + k] ^ ycode(y);
            u[y * W + k] = cur ^ enc_word(y);
            prev = cur;
        }
    }
    __syncthreads();
}

// ---- u -> slopes (HBM): every word independently, periodic in x and y -----------------------------------------
__device__ __forceinline__ void resident_store(uint32_t* __restrict__ planeX, uint32_t* __restrict__ planeY, uint32_t L,
                                               uint32_t W, const uint32_t* __restrict__ u, uint32_t tid, uint32_t nthr) {
    const uint32_t n = L * W;
    for (uint32_t i = tid; i < n; i += nthr) {
        const uint32_t y = i / W, k = i - y * W;
        const uint32_t yb = (y == 0u) ? L - 1u : y - 1u;
        const uint32_t kp = (k == 0u) ? W - 1u : k - 1u;
        const uint32_t cur = u[i] ^ enc_word(y);
        const uint32_t below = u[yb * W + k] ^ enc_word(yb);
        const uint32_t left = __funnelshift_l(u[y * W + kp] ^ enc_word(y), cur, 1);
        planeY[i] = cur ^ below ^ ycode(y);           // sigma_y(.,y) = h1(y) ^ h1(y-1) ^ ycode(y)
        planeX[i] = cur ^ left ^ ycode(y);            // sigma_x(x,y) = h1(x) ^ h1(x-1) ^ h0(x,y)
    }
}

// ---- one attempt of the thread-per-tile variant on the shared lattice bitmap -----------------------------------
template <bool GENERAL>
__device__ __forceinline__ void resident_attempt(uint32_t* u, uint32_t L, uint32_t W, uint32_t X, uint32_t Y,
                                                 uint32_t accept_word, const ResidentParams& P, uint32_t& n_dep,
                                                 uint32_t& n_rem, int32_t& dh00) {
    const uint32_t wi = X >> 5;
    uint32_t* row = u + Y * W;
    const uint32_t wo = row[wi], wp = row[(wi - 1u) & (W - 1u)], wn = row[(wi + 1u) & (W - 1u)];
    const uint32_t wu = u[((Y + 1u) & (L - 1u)) * W + wi], wd = u[((Y - 1u) & (L - 1u)) * W + wi];
    uint32_t mn, mx;
    minmax_words(wo, wp, wn, wu, wd, mn, mx);
    const uint32_t bit = 1u << (X & 31u);
    uint32_t md = mn & bit, mr = 0u;
    if (GENERAL) {
        md = ((uint64_t)accept_word < P.thr_p) ? md : 0u;
        mr = ((uint64_t)accept_word < P.thr_q) ? (mx & bit) : 0u;
    }
    if (md | mr) atomicXor(row + wi, md | mr);
    n_dep += md ? 1u : 0u;
    n_rem += mr ? 1u : 0u;
    if ((X | Y) == 0u) dh00 += md ? 2 : (mr ? -2 : 0);
}

// shared-memory words per warp of the cooperative variant: 128 site words + 256 accept words of a 256-step group
constexpr int KPZ_COOP_WARP_WORDS = 128 + 256;

// GENERAL = false: p = 1, q = 0 (the accept stream is never evaluated: bit-identical, R12).
template <int T, bool GENERAL, bool COOP>
__global__ void __launch_bounds__(1024) kpz_resident_kernel(const ResidentParams P) {
    using Geo = TileGeom<T>;
    constexpr uint32_t TT = (uint32_t)(T * T);
    constexpr uint32_t ACCEPT = 0x80000000u;
    extern __shared__ uint32_t smem[];
    const uint32_t L = P.L, W = P.W, LW = L * W;
    const uint32_t tid = threadIdx.x, nthr = blockDim.x;
    const uint32_t g0 = blockIdx.x * P.G;                         // first replica of this CTA
    const uint32_t ng = min(P.G, P.R - g0);                       // replicas of this CTA

    // ---- load ----
    for (uint32_t g = 0; g < ng; ++g) {
        const uint32_t* planeX = P.lattice + (size_t)(g0 + g) * 2u * P.plane_words;
        resident_load(planeX, planeX + P.plane_words, L, W, smem + g * LW, tid, nthr);
    }
    uint32_t n_dep = 0, n_rem = 0;
    int32_t dh00 = 0;

    if constexpr (!COOP) {
        // ---- one thread per tile ----
        const uint32_t items = ng * P.tpc;
        for (uint32_t mi = 0; mi < P.n_mcs; ++mi) {
            const uint32_t m = P.m0 + mi;
            for (uint32_t slot = 0; slot < 4u; ++slot) {
                for (uint32_t it = tid; it < items; it += nthr) {
                    const uint32_t g = it / P.tpc, wl = it - g * P.tpc;
                    const uint32_t replica = g0 + g;
                    uint32_t ox, oy, perm;
                    resident_draw<T>(P.key, m, replica, ox, oy, perm);
                    const uint32_t colour = (perm >> (2u * slot)) & 3u;
                    const uint32_t j = wl / P.HN, i = wl - j * P.HN;
                    const uint32_t tx = 2u * i + (colour & 1u), ty = 2u * j + (colour >> 1);
                    const uint32_t X0 = ox + tx * T, Y0 = oy + ty * T, tile_id = ty * P.NT + tx;
                    uint32_t* u = smem + g * LW;
                    uint32_t nd = 0, nr = 0;
                    int32_t dh = 0;
                    uint4 cur = philox4x32_10(0u, tile_id, m, replica, P.key);
#pragma unroll 1
                    for (uint32_t c = 0; c < TT / 8u; ++c) {
                        const uint4 nxt = philox4x32_10(c + 1u, tile_id, m, replica, P.key);   // one call ahead
                        uint4 a0 = make_uint4(0u, 0u, 0u, 0u), a1 = a0;
                        if (GENERAL) {
                            a0 = philox4x32_10((2u * c) | ACCEPT, tile_id, m, replica, P.key);
                            a1 = philox4x32_10((2u * c + 1u) | ACCEPT, tile_id, m, replica, P.key);
                        }
                        const uint32_t sw[8] = {cur.x, cur.x * TT, cur.y, cur.y * TT, cur.z, cur.z * TT, cur.w, cur.w * TT};
                        const uint32_t aw[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
#pragma unroll
                        for (int s = 0; s < 8; ++s) {
                            const uint32_t idx = sw[s] >> (32 - 2 * Geo::LOG2T);
                            const uint32_t X = (X0 + (idx & (uint32_t)(T - 1))) & (L - 1u);
                            const uint32_t Y = (Y0 + (idx >> Geo::LOG2T)) & (L - 1u);
                            resident_attempt<GENERAL>(u, L, W, X, Y, aw[s], P, nd, nr, dh);
                        }
                        cur = nxt;
                    }
                    if (nd | nr | (uint32_t)dh) {
                        unsigned long long* st = P.stats + (size_t)replica * 4u;
                        if (nd) atomicAdd(st + 0, (unsigned long long)nd);
                        if (nr) atomicAdd(st + 1, (unsigned long long)nr);
                        if (dh) atomicAdd(st + 2, (unsigned long long)(long long)dh);
                    }
                }
                __syncthreads();
            }
        }
    } else {
        // ---- one warp per tile, G = 1 ----
        const uint32_t replica = g0;
        uint32_t* u = smem;
        uint32_t* Mn = smem + LW;
        uint32_t* Mx = Mn + LW;                                   // allocated only when GENERAL
        const uint32_t lane = tid & 31u, warp = tid >> 5, nwarps = nthr >> 5;
        uint32_t* rng = smem + (GENERAL ? 3u : 2u) * LW + warp * KPZ_COOP_WARP_WORDS;
        uint32_t* acc = rng + 128;
        // minima / maxima bitmaps of the whole lattice
        for (uint32_t i = tid; i < LW; i += nthr) {
            const uint32_t y = i / W, k = i - y * W;
            uint32_t mn, mx;
            minmax_words(u[i], u[y * W + ((k - 1u) & (W - 1u))], u[y * W + ((k + 1u) & (W - 1u))],
                         u[((y + 1u) & (L - 1u)) * W + k], u[((y - 1u) & (L - 1u)) * W + k], mn, mx);
            Mn[i] = mn;
            if (GENERAL) Mx[i] = mx;
        }
        __syncthreads();
        for (uint32_t mi = 0; mi < P.n_mcs; ++mi) {
            const uint32_t m = P.m0 + mi;
            uint32_t ox, oy, perm;
            resident_draw<T>(P.key, m, replica, ox, oy, perm);
            for (uint32_t slot = 0; slot < 4u; ++slot) {
                const uint32_t colour = (perm >> (2u * slot)) & 3u;
                for (uint32_t wl = warp; wl < P.tpc; wl += nwarps) {
                    const uint32_t j = wl / P.HN, i = wl - j * P.HN;
                    const uint32_t tx = 2u * i + (colour & 1u), ty = 2u * j + (colour >> 1);
                    const uint32_t X0 = ox + tx * T, Y0 = oy + ty * T, tile_id = ty * P.NT + tx;
                    for (uint32_t gb = 0; gb < TT; gb += 256u) {
                        // the Philox calls of the next 256 steps: lane l makes site call gb/8 + l (8 steps) and
                        // accept calls gb/4 + l, gb/4 + 32 + l (4 steps each)
                        __syncwarp();
                        if (gb + 8u * lane < TT) {
                            const uint4 q = philox4x32_10((gb >> 3) + lane, tile_id, m, replica, P.key);
                            *reinterpret_cast<uint4*>(rng + 4u * lane) = q;
                        }
                        if (GENERAL) {
#pragma unroll
                            for (uint32_t h = 0; h < 2u; ++h) {
                                if (gb + 4u * (lane + 32u * h) < TT) {
                                    const uint4 q = philox4x32_10(((gb >> 2) + lane + 32u * h) | ACCEPT, tile_id, m, replica, P.key);
                                    *reinterpret_cast<uint4*>(acc + 4u * (lane + 32u * h)) = q;
                                }
                            }
                        }
                        __syncwarp();
                        const uint32_t nb = min(8u, (TT - gb + 31u) >> 5);
                        for (uint32_t b = 0; b < nb; ++b) {
                            const uint32_t s = gb + 32u * b + lane;
                            const bool live = s < TT;
                            uint32_t wsite = rng[16u * b + (lane >> 1)];
                            if (lane & 1u) wsite *= TT;
                            const uint32_t idx = wsite >> (32 - 2 * Geo::LOG2T);
                            const uint32_t X = (X0 + (idx & (uint32_t)(T - 1))) & (L - 1u);
                            const uint32_t Y = (Y0 + (idx >> Geo::LOG2T)) & (L - 1u);
                            const uint32_t mw = Y * W + (X >> 5), bb = X & 31u;
                            bool okp = true, okq = false;
                            if (GENERAL) {
                                const uint32_t a = acc[32u * b + lane];
                                okp = (uint64_t)a < P.thr_p;
                                okq = (uint64_t)a < P.thr_q;
                            }
                            bool is_min = live && okp && ((Mn[mw] >> bb) & 1u);
                            bool is_max = GENERAL && live && okq && ((Mx[mw] >> bb) & 1u);
                            uint32_t cand = __ballot_sync(0xFFFFFFFFu, is_min || is_max);
                            while (cand) {
                                const uint32_t c = (uint32_t)__ffs((int)cand) - 1u;
                                const uint32_t Xc = __shfl_sync(0xFFFFFFFFu, X, c), Yc = __shfl_sync(0xFFFFFFFFu, Y, c);
                                const uint32_t wic = Xc >> 5, bc = Xc & 31u;
                                const uint32_t was_min = __shfl_sync(0xFFFFFFFFu, (uint32_t)is_min, c);
                                if (lane == 0u) {
                                    atomicXor(u + Yc * W + wic, 1u << bc);
                                    if (was_min) { ++n_dep; if ((Xc | Yc) == 0u) dh00 += 2; }
                                    else { ++n_rem; if ((Xc | Yc) == 0u) dh00 -= 2; }
                                }
                                __syncwarp();
                                // the five words of M that hold the sites within distance 1 of the flip: lane 0..4 =
                                // (Yc, wic), (Yc, wic-1), (Yc, wic+1), (Yc-1, wic), (Yc+1, wic); only the N5 bits change
                                if (lane < 5u) {
                                    const uint32_t yy = (lane == 3u) ? ((Yc - 1u) & (L - 1u)) : (lane == 4u) ? ((Yc + 1u) & (L - 1u)) : Yc;
                                    const uint32_t kk = (lane == 1u) ? ((wic - 1u) & (W - 1u)) : (lane == 2u) ? ((wic + 1u) & (W - 1u)) : wic;
                                    uint32_t nmask;
                                    if (lane == 0u) nmask = (1u << bc) | ((1u << bc) << 1) | ((1u << bc) >> 1);
                                    else if (lane == 1u) nmask = (bc == 0u) ? 0x80000000u : 0u;
                                    else if (lane == 2u) nmask = (bc == 31u) ? 1u : 0u;
                                    else nmask = 1u << bc;
                                    if (nmask) {
                                        uint32_t mn, mx;
                                        minmax_words(u[yy * W + kk], u[yy * W + ((kk - 1u) & (W - 1u))], u[yy * W + ((kk + 1u) & (W - 1u))],
                                                     u[((yy + 1u) & (L - 1u)) * W + kk], u[((yy - 1u) & (L - 1u)) * W + kk], mn, mx);
                                        const uint32_t dn = (Mn[yy * W + kk] ^ mn) & nmask;
                                        if (dn) atomicXor(Mn + yy * W + kk, dn);
                                        if (GENERAL) {
                                            const uint32_t dx = (Mx[yy * W + kk] ^ mx) & nmask;
                                            if (dx) atomicXor(Mx + yy * W + kk, dx);
                                        }
                                    }
                                }
                                __syncwarp();
                                // later lanes re-read their bit (only sites next to the flip can have changed)
                                const bool later = lane > c;
                                is_min = later && live && okp && ((Mn[mw] >> bb) & 1u);
                                is_max = GENERAL && later && live && okq && ((Mx[mw] >> bb) & 1u);
                                cand = __ballot_sync(0xFFFFFFFFu, is_min || is_max);
                            }
                        }
                    }
                }
                __syncthreads();
            }
        }
        if (lane == 0u && (n_dep | n_rem | (uint32_t)dh00)) {
            unsigned long long* st = P.stats + (size_t)replica * 4u;
            if (n_dep) atomicAdd(st + 0, (unsigned long long)n_dep);
            if (n_rem) atomicAdd(st + 1, (unsigned long long)n_rem);
            if (dh00) atomicAdd(st + 2, (unsigned long long)(long long)dh00);
        }
    }

    // ---- store ----
    __syncthreads();
    for (uint32_t g = 0; g < ng; ++g) {
        uint32_t* planeX = P.lattice + (size_t)(g0 + g) * 2u * P.plane_words;
        resident_store(planeX, planeX + P.plane_words, L, W, smem + g * LW, tid, nthr);
    }
}

}  // namespace kpz
