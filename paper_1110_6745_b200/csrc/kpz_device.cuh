// kpz_device.cuh -- device code of the B200-native octahedron-KPZ hot path (sm_100a).
//
// Kernels:
//   kpz_update_kernel<T,...>   steps a2-a6 of SURVEY 8(a): tile + halo staged into shared memory as one height bit
//                              per site, T*T sequential Philox-driven attempts per tile (eq. 2), write-back.
//   kpz_resident_kernel<T,...> the same steps with the packed lattice held in shared memory for all MCS of a call.
// The measurement, flat-start, spectrum and parity / checkpoint kernels are in kpz_aux_kernels.cuh.
//
// Nothing here is shared with the CPU checker of the tests (own Philox, own rule, own height walk).
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
    unsigned long long* stats;     // device: [R][4] = deposits, removals, h00 (two's complement), attempts made under S7
    uint64_t plane_words;          // L*L/32
    uint64_t total_items;          // R * HN*HN  (tiles of one colour over all replicas)
    uint64_t thr_p, thr_q;         // accept iff (uint64)word < thr
    uint32_t tp_incl, tq_incl;     // thr - 1 (MODE 1: both thresholds >= 1, accept iff word <= thr - 1)
    uint32_t L, NT, HN;            // lattice edge, tiles per edge, NT/2
    uint32_t W;                    // L/32: words per bit-line
    uint32_t tiles_per_colour;     // HN * HNy
    // A handle may hold one SLAB of the lattice: `rows` consecutive rows starting at global
    // tile row ty0 (storage row 0 = global row ty0 * T), tile rows ty0 .. ty0 + 2 HNy - 1 of the shifted frame.  The
    // whole lattice is the case rows = ywrap = L, ty0 = 0, HNy = HN.
    uint32_t HNy;                  // tile rows of one colour in this launch
    uint32_t ty0;                  // first global tile row of the stored rows
    uint32_t ywrap;                // row index at which the stored rows wrap around: L, or 0xFFFFFFFF for a slab (never)
    // A launch may cover only the tile-row pairs j0 .. j0 + HNy - 1 of a whole lattice (kpz_step_host_overlapped runs the
    // colour passes slab by slab while the rest of the lattice is still in flight); a tile row index >= tywrap wraps.
    uint32_t j0;                   // first tile-row pair of this launch (0: from the first)
    uint32_t tywrap;               // NT for a whole lattice, 0xFFFFFFFF for a slab
    uint32_t blocked;              // 1: 8x4 lane blocking of tiles (HN % 8 == 0), 0: linear
    uint32_t m;                    // MCS index (number of completed MCS)
    uint32_t slot;                 // 0..3: which entry of the colour order this launch executes
    uint32_t sub;                  // sub-sweep index j (S6): counter word c0 of the global draw
    uint32_t call_begin, call_end; // site calls [call_begin, call_end) of every tile: steps 8*call_begin .. 8*call_end
    const unsigned long long* pthr; // S7: device table, pthr[i] = floor(2^32 P(n <= pk_min + i)), pn entries
    uint32_t pn, pk_min;
    PhiloxKey key;
};

// Global draw of MCS m for one replica: offset (multiples of 4 sites) and colour order.
// DESIGN.md "Schedule" S2.  Returns the colour processed in `slot`.
template <int T>
__device__ __forceinline__ void global_draw(const UpdateParams& P, uint32_t sub, uint32_t replica, uint32_t& ox, uint32_t& oy,
                                            uint32_t& colour) {
    const uint4 G = philox4x32_10(sub, 0xFFFFFFFFu, P.m, replica, P.key);
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
// Update kernel.  One THREAD owns one tile for all of its T*T sequential attempts (program order = schedule
// order S3).  In shared memory the tile is NOT kept as slopes but as ONE bit per site, the high bit h1 of the
// height modulo 4:
//   in-tile heights are taken relative to an anchor of the right parity, h = 2*h1 + h0 (mod 4) with the low bit
//   h0(lx,ly) = (lx+ly) & 1 fixed for ever (every step of the surface is +-1, every flip is +-2).  Then
//     local minimum at a site with parity pi  <=>  all four neighbours have h1 == own_h1 ^ pi,
//     local maximum                           <=>  all four neighbours have h1 != own_h1 ^ pi,
//     a flip in either direction              <=>  XOR of the site's own h1 bit  (one shared-memory reduction).
// What is stored is u = h1 ^ E(x,y) (enc_word / enc_narrow below), which makes the two tests independent of pi.
// Rows ly = -1 .. T (row index r = ly+1) hold the tile plus its 1-site halo on all four sides (the -x / -y
// halos carry sigma_x(x0,.) / sigma_y(.,y0), which belong to the tile's own sites; the +x / +y halos are the slopes
// on the inactive neighbours that a border update changes).
//   T >= 32: a row is WPL = T/32 own words (bit lx&31 of word lx>>5) followed by one halo word H_r with
//            bit 0 = h1(T, ly) and bit 31 = h1(-1, ly+1): the word before / after any own word then supplies the
//            left / right neighbour of its bit 0 / bit 31 through one funnel shift -- no special case at the border.
//   T <  32: a row is one word, bit p = lx+1 (bit 0 and bit T+1 are the halos).
// Word w of thread t sits at smem[w * NTHR + t]: every thread stays in its own bank (conflict-free for any
// access pattern) and threads never share data: no barrier anywhere in the kernel.
// ------------------------------------------------------------------------------------------------------------
template <int T>
struct TileGeom {
    static constexpr int LOG2T = (T == 4) ? 2 : (T == 8) ? 3 : (T == 16) ? 4 : (T == 32) ? 5 : 6;
    static constexpr bool WIDE = (T >= 32);
    static constexpr int WPL = WIDE ? T / 32 : 1;      // own words per row
    static constexpr int WPR = WIDE ? WPL + 1 : 1;     // words per row in shared memory
    static constexpr int ROWS = T + 2;                 // ly = -1 .. T
    static constexpr int PAD = WIDE ? 1 : 0;           // word "before" row 0 (never meaningful, keeps addresses valid)
    static constexpr int WORDS = PAD + ROWS * WPR;     // per tile
    static constexpr uint32_t LINE_MASK = (T >= 32) ? 0xFFFFFFFFu : ((1u << (T & 31)) - 1u);
};

// rows fetched per batch while staging: all loads of a batch are issued before the first dependent use, so one
// thread keeps tens of requests in flight.  N divides T+1.
template <int T>
struct StageBatch {
    static constexpr int N = (T == 64) ? 13 : (T == 32) ? 11 : (T + 1);
};

// sigma_y(.,ly) = row(ly) ^ row(ly-1) ^ ycode(ly) and back (own columns, bit j <-> parity of lx):
// h1(ly) = h1(ly-1) ^ XNOR(sigma_y(ly), h0(.,ly-1)),  h0(lx,ly-1) = (lx+ly-1)&1.
__device__ __forceinline__ uint32_t ycode(uint32_t ly) { return 0xAAAAAAAAu ^ (0u - (ly & 1u)); }

// inclusive prefix XOR over the 32 bits of a word
__device__ __forceinline__ uint32_t prefix_xor32(uint32_t t) {
    t ^= t << 1; t ^= t << 2; t ^= t << 4; t ^= t << 8; t ^= t << 16;
    return t;
}

// Parity-free encoding of the T >= 32 tile: shared memory holds u = h1 ^ E with
//   E(x,y) = ((x + (y&1)) >> 1 & 1) ^ (y >> 1 & 1)      (period 4 in x and y; words start at multiples of 32),
// chosen so that the test of eq. 2 needs no parity word:
//   local minimum  <=>  u(x+1,y) == u, u(x-1,y) != u, u(x,y+1) == u, u(x,y-1) != u;   local maximum: all four reversed.
// enc_word(ly): E over the 32 columns of an own word of row ly;  enc_halo(ly): E of the two used bits of the halo
// word H_ly (bit 0 = column T of row ly, bit 31 = column -1 of row ly+1).  ly = -1 is 0xFFFFFFFF (== 3 mod 4).
__device__ __forceinline__ uint32_t enc_word(uint32_t ly) {
    return ((ly & 1u) ? 0x66666666u : 0xCCCCCCCCu) ^ (0u - ((ly >> 1) & 1u));
}
// T < 32 (bit p of a row word is column p - 1): the same pattern one bit up, E has period 4 in x
__device__ __forceinline__ uint32_t enc_narrow(uint32_t ly) { return __funnelshift_l(enc_word(ly), enc_word(ly), 1); }
__device__ __forceinline__ uint32_t enc_halo(uint32_t ly) {
    const uint32_t y1 = ly + 1u;
    return ((ly >> 1) & 1u) | ((((y1 & 1u) ^ 1u) ^ ((y1 >> 1) & 1u)) << 31);
}

// N running pointers into consecutive rows of the bit-planes (periodic in y): one 64-bit add per pointer and row
// instead of a multiply and a scaled add per access.
template <int N>
struct RowPtrs {
    uint32_t* p[N];
    uint32_t g;
    __device__ __forceinline__ void next(uint32_t L, uint32_t W) {
        ptrdiff_t st = (ptrdiff_t)W;
        if (++g == L) {
            g = 0u;
            st -= (ptrdiff_t)L * (ptrdiff_t)W;
        }
#pragma unroll
        for (int k = 0; k < N; ++k) p[k] += st;
    }
};

// ---- a2: stage tile + halo, slopes (HBM) -> height bits (shared memory), T >= 32 -----------------------------
template <int T, int NTHR, int NB = StageBatch<T>::N>
__device__ __forceinline__ void stage_in_wide(const uint32_t* __restrict__ planeX, const uint32_t* __restrict__ planeY,
                                              uint32_t L, uint32_t W, uint32_t x0, uint32_t y0, uint32_t* __restrict__ sm) {
    using G = TileGeom<T>;
    constexpr int WPL = G::WPL;
    const uint32_t s = x0 & 31u;
    uint32_t idx[WPL + 1];
    idx[0] = x0 >> 5;
#pragma unroll
    for (int k = 1; k <= WPL; ++k) idx[k] = (idx[k - 1] + 1u == W) ? 0u : idx[k - 1] + 1u;

    // row ly = 0 from sigma_x(.,y0): h1(0,0) = 0 is the anchor, h1(lx,0) = XOR_{l=1..lx} XNOR(sigma_x(l), h0(l-1,0))
    uint32_t prev[WPL];
    {
        const uint32_t* line = planeX + (size_t)y0 * W;
        uint32_t raw[WPL + 1];
#pragma unroll
        for (int k = 0; k <= WPL; ++k) raw[k] = line[idx[k]];
        uint32_t carry = 0u;
#pragma unroll
        for (int k = 0; k < WPL; ++k) {
            uint32_t t = __funnelshift_r(raw[k], raw[k + 1], s) ^ 0xAAAAAAAAu;   // h0(l-1,0) = 1 for even l
            if (k == 0) t &= ~1u;
            t = prefix_xor32(t) ^ carry;
            carry = 0u - (t >> 31);
            prev[k] = t;
        }
    }
    uint32_t pendingH = 0u;    // halo word of the previous row: bit 0 already holds its +x halo
    // words idx[0..WPL] of plane Y and words idx[0], idx[WPL] of plane X, row by row from y0
    RowPtrs<WPL + 3> rp;
    rp.g = y0;
#pragma unroll
    for (int k = 0; k <= WPL; ++k) rp.p[k] = const_cast<uint32_t*>(planeY) + (size_t)y0 * W + idx[k];
    rp.p[WPL + 1] = const_cast<uint32_t*>(planeX) + (size_t)y0 * W + idx[0];
    rp.p[WPL + 2] = const_cast<uint32_t*>(planeX) + (size_t)y0 * W + idx[WPL];
#pragma unroll 1
    for (int l0 = 0; l0 <= T; l0 += NB) {
        uint32_t ry[NB][WPL + 1], rx[NB][2];
#pragma unroll
        for (int b = 0; b < NB; ++b) {
#pragma unroll
            for (int k = 0; k <= WPL; ++k) ry[b][k] = *rp.p[k];
            rx[b][0] = *rp.p[WPL + 1];
            rx[b][1] = *rp.p[WPL + 2];
            rp.next(L, W);
        }
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const uint32_t ly = (uint32_t)(l0 + b);
            const uint32_t r = ly + 1u;
            uint32_t cur[WPL];
            const uint32_t yc = ycode(ly);
            if (b == 0 && l0 == 0) {
                // rows -1 and 0:  row(-1) = row(0) ^ sigma_y(.,0) ^ ycode(0)
#pragma unroll
                for (int k = 0; k < WPL; ++k) {
                    const uint32_t yv = __funnelshift_r(ry[b][k], ry[b][k + 1], s);
                    cur[k] = prev[k];
                    sm[(G::PAD + k) * NTHR] = prev[k] ^ yv ^ yc ^ enc_word(0xFFFFFFFFu);
                }
            } else {
#pragma unroll
                for (int k = 0; k < WPL; ++k) {
                    const uint32_t yv = __funnelshift_r(ry[b][k], ry[b][k + 1], s);
                    cur[k] = prev[k] ^ yv ^ yc;
                }
            }
#pragma unroll
            for (int k = 0; k < WPL; ++k) sm[(G::PAD + r * G::WPR + k) * NTHR] = cur[k] ^ enc_word(ly);
            if (ly < (uint32_t)T) {
                // halos of this row from sigma_x(x0, y) and sigma_x(x0+T, y):  h1(A) = h1(B) ^ sigma ^ (ly & 1)
                const uint32_t bL = (rx[b][0] >> s) & 1u, bR = (rx[b][1] >> s) & 1u;
                const uint32_t hL = (cur[0] ^ bL ^ ly) & 1u;
                const uint32_t hR = ((cur[WPL - 1] >> 31) ^ bR ^ ly) & 1u;
                sm[(G::PAD + (r - 1u) * G::WPR + WPL) * NTHR] = (pendingH | (hL << 31)) ^ enc_halo(ly - 1u);
                pendingH = hR;
            } else {
                sm[(G::PAD + (r - 1u) * G::WPR + WPL) * NTHR] = pendingH ^ enc_halo(ly - 1u);
            }
#pragma unroll
            for (int k = 0; k < WPL; ++k) prev[k] = cur[k];
        }
    }
}

// ---- a5: write back, height bits -> slopes, T >= 32.  The first and last word of a row segment are shared with
// the (inactive, other-colour) neighbour tiles: re-read and merged.  No other thread of the launch touches
// these words.
template <int T, int NTHR, int NB = StageBatch<T>::N, bool DEAD = false>
__device__ __forceinline__ void stage_out_wide(uint32_t* __restrict__ planeX, uint32_t* __restrict__ planeY, uint32_t L,
                                               uint32_t W, uint32_t x0, uint32_t y0, const uint32_t* __restrict__ sm) {
    using G = TileGeom<T>;
    constexpr int WPL = G::WPL;
    const uint32_t s = x0 & 31u;
    const uint32_t lowmask = (1u << s) - 1u;            // bits below the segment start
    const uint32_t lowmask1 = lowmask | (1u << s);      // ... and the bit that holds sigma_x(x0+T)
    uint32_t idx[WPL + 1];
    idx[0] = x0 >> 5;
#pragma unroll
    for (int k = 1; k <= WPL; ++k) idx[k] = (idx[k - 1] + 1u == W) ? 0u : idx[k - 1] + 1u;
    // edge words (re-read) and all words (stored) of both planes, row by row from y0:
    // ld: Y idx[0], Y idx[WPL], X idx[0], X idx[WPL];   st: Y idx[0..WPL], X idx[0..WPL]
    RowPtrs<4> ld;
    RowPtrs<2 * (WPL + 1)> st;
    ld.g = st.g = y0;
    ld.p[0] = planeY + (size_t)y0 * W + idx[0];
    ld.p[1] = planeY + (size_t)y0 * W + idx[WPL];
    ld.p[2] = planeX + (size_t)y0 * W + idx[0];
    ld.p[3] = planeX + (size_t)y0 * W + idx[WPL];
#pragma unroll
    for (int k = 0; k <= WPL; ++k) {
        st.p[k] = planeY + (size_t)y0 * W + idx[k];
        st.p[WPL + 1 + k] = planeX + (size_t)y0 * W + idx[k];
    }
#pragma unroll 1
    for (int l0 = 0; l0 <= T; l0 += NB) {
        uint32_t ex[NB][2], ey[NB][2];
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            ey[b][0] = *ld.p[0];
            ey[b][1] = *ld.p[1];
            ex[b][0] = *ld.p[2];
            ex[b][1] = *ld.p[3];
            ld.next(L, W);
        }
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const uint32_t ly = (uint32_t)(l0 + b);
            const uint32_t r = ly + 1u;
            uint32_t* const* ly_ = st.p;               // *ly_[k] = word idx[k] of this row of plane Y
            uint32_t* const* lx_ = st.p + (WPL + 1);   // ... of plane X
            uint32_t cur[WPL], below[WPL];
#pragma unroll
            for (int k = 0; k < WPL; ++k) {
                cur[k] = sm[(G::PAD + r * G::WPR + k) * NTHR] ^ enc_word(ly);
                below[k] = sm[(G::PAD + (r - 1u) * G::WPR + k) * NTHR] ^ enc_word(ly - 1u);
            }
            // sigma_y(.,ly): T bits at bit offset x0
            {
                const uint32_t yc = ycode(ly);
                uint32_t v[WPL];
#pragma unroll
                for (int k = 0; k < WPL; ++k) v[k] = cur[k] ^ below[k] ^ yc;
                if (DEAD) {
                    // S5: every tile is active, the edge words are shared with running neighbours: apply only this
                    // tile's own changed bits, atomically; rows 0..T-1 only
                    if (ly < (uint32_t)T) {
                        const uint32_t d0 = (ey[b][0] ^ (v[0] << s)) & ~lowmask;
                        if (d0) atomicXor(ly_[0], d0);
#pragma unroll
                        for (int k = 1; k < WPL; ++k) *ly_[k] = __funnelshift_l(v[k - 1], v[k], s);
                        const uint32_t d1 = (ey[b][1] ^ __funnelshift_l(v[WPL - 1], 0u, s)) & lowmask;
                        if (d1) atomicXor(ly_[WPL], d1);
                    }
                } else {
                    *ly_[0] = (ey[b][0] & lowmask) | (v[0] << s);
#pragma unroll
                    for (int k = 1; k < WPL; ++k) *ly_[k] = __funnelshift_l(v[k - 1], v[k], s);
                    if (s != 0u) *ly_[WPL] = (ey[b][1] & ~lowmask) | __funnelshift_l(v[WPL - 1], 0u, s);
                }
            }
            // sigma_x(.,ly): T+1 bits (lx = 0..T) at bit offset x0; rows 0..T-1 only
            if (ly < (uint32_t)T) {
                const uint32_t hprev = sm[(G::PAD + (r - 1u) * G::WPR + WPL) * NTHR] ^ enc_halo(ly - 1u);   // bit 31 = h1(-1, ly)
                const uint32_t hcur = sm[(G::PAD + r * G::WPR + WPL) * NTHR] ^ enc_halo(ly);               // bit 0  = h1(T, ly)
                const uint32_t xc = ycode(ly);      // bit j = (j + ly) & 1 = h0(lx, ly)
                uint32_t v[WPL];
#pragma unroll
                for (int k = 0; k < WPL; ++k) {
                    const uint32_t left = __funnelshift_l(k == 0 ? hprev : cur[k - 1], cur[k], 1);
                    v[k] = cur[k] ^ left ^ xc;
                }
                const uint32_t bitT = (hcur ^ (cur[WPL - 1] >> 31) ^ ly) & 1u;          // (T + ly) & 1 = ly & 1
                if (DEAD) {
                    // S5: bits lx = 0..T-1 only (bit T is sigma_x of the right neighbour's own column 0)
                    const uint32_t d0 = (ex[b][0] ^ (v[0] << s)) & ~lowmask;
                    if (d0) atomicXor(lx_[0], d0);
#pragma unroll
                    for (int k = 1; k < WPL; ++k) *lx_[k] = __funnelshift_l(v[k - 1], v[k], s);
                    const uint32_t d1 = (ex[b][1] ^ __funnelshift_l(v[WPL - 1], 0u, s)) & lowmask;
                    if (d1) atomicXor(lx_[WPL], d1);
                } else {
                    *lx_[0] = (ex[b][0] & lowmask) | (v[0] << s);
#pragma unroll
                    for (int k = 1; k < WPL; ++k) *lx_[k] = __funnelshift_l(v[k - 1], v[k], s);
                    *lx_[WPL] = (ex[b][1] & ~lowmask1) | __funnelshift_l(v[WPL - 1], 0u, s) | (bitT << s);
                }
            }
            st.next(L, W);
        }
    }
}

// ---- T < 32: a row is one word, bit p = lx+1. -------------------------------------------------------------------
// T < 32 staging: the rows of the tile are fetched (or re-read) in batches of up to 9 rows of two words per plane
// before the first dependent use, so the global-memory latency is paid once per batch and not once per row.
template <int T>
struct NarrowBatch {
    static constexpr int N = (T + 1 <= 9) ? T + 1 : 9;
};

template <int T, int NTHR>
__device__ __forceinline__ void stage_in_narrow(const uint32_t* __restrict__ planeX, const uint32_t* __restrict__ planeY,
                                                uint32_t L, uint32_t W, uint32_t x0, uint32_t y0, uint32_t* __restrict__ sm) {
    constexpr uint32_t MT = (1u << T) - 1u;          // T bits
    constexpr uint32_t MT1 = (2u << T) - 1u;         // T+1 bits
    constexpr uint32_t MROW = (4u << T) - 1u;        // T+2 bits of a row word (halo, T columns, halo)
    constexpr int R = T + 1, NB = NarrowBatch<T>::N;
    const uint32_t a = x0 >> 5;
    const uint32_t a1 = (a + 1u == W) ? 0u : a + 1u;
    uint32_t g = y0;
    size_t row = (size_t)y0 * W;
    uint32_t prev = 0u;                               // h1 of the previous row, bit lx
#pragma unroll 1
    for (int r0 = 0; r0 < R; r0 += NB) {
        uint32_t yl[NB], yh[NB], xl[NB], xh[NB];
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            if (r0 + b < R) {
                yl[b] = planeY[row + a];
                yh[b] = planeY[row + a1];
                if (r0 + b < T) {
                    xl[b] = planeX[row + a];
                    xh[b] = planeX[row + a1];
                }
                row += W;
                if (++g == L) { g = 0u; row = 0; }
            }
        }
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const int r = r0 + b;
            if (r < R) {
                const uint32_t ly = (uint32_t)r;
                const uint32_t yv = __funnelshift_r(yl[b], yh[b], x0) & MT;
                const uint32_t xv = (r < T) ? (__funnelshift_r(xl[b], xh[b], x0) & MT1) : 0u;
                const uint32_t yc = ycode(ly) & MT;
                uint32_t cur;
                if (r == 0) {
                    cur = prefix_xor32((xv ^ 0xAAAAAAAAu) & MT & ~1u) & MT;
                    sm[0] = (((cur ^ yv ^ yc) & MT) << 1) ^ (enc_narrow(0xFFFFFFFFu) & MROW);   // row -1: own columns only
                } else {
                    cur = prev ^ yv ^ yc;
                }
                uint32_t word = cur << 1;
                if (r < T) {
                    const uint32_t hL = (cur ^ xv ^ ly) & 1u;
                    const uint32_t hR = ((cur >> (T - 1)) ^ (xv >> T) ^ ly) & 1u;
                    word |= hL | (hR << (T + 1));
                }
                sm[(ly + 1u) * NTHR] = word ^ (enc_narrow(ly) & MROW);
                prev = cur;
            }
        }
    }
}

// Writes the bits selected by `mask` (in segment coordinates) of `seg`; the segment sits at bit offset o (a multiple
// of 4, it may span two words) and its two words were read before as (lo, hi).  Two same-colour tiles may share a
// 32-bit word (and, for T = 4, a byte) when T < 32, so only the CHANGED bits are applied, with an XOR reduction:
// every bit of a segment belongs to exactly one active tile, hence old ^ new on its own bits is exact (and stays so
// when the words were read before other tiles' reductions landed).
__device__ __forceinline__ void store_bits_pre(uint32_t* __restrict__ plo, uint32_t* __restrict__ phi, uint32_t o, uint32_t mask,
                                               uint32_t seg, uint32_t lo, uint32_t hi) {
    const uint32_t old = __funnelshift_r(lo, hi, o) & mask;
    const uint32_t d = old ^ (seg & mask);
    const uint32_t s = o & 31u;
    const uint32_t dlo = d << s;
    const uint32_t dhi = __funnelshift_l(d, 0u, s);      // d >> (32 - s), 0 for s = 0
    if (dlo) atomicXor(plo, dlo);
    if (dhi) atomicXor(phi, dhi);
}

template <int T, int NTHR, bool DEAD>
__device__ __forceinline__ void stage_out_narrow(uint32_t* __restrict__ planeX, uint32_t* __restrict__ planeY, uint32_t L,
                                                 uint32_t W, uint32_t x0, uint32_t y0, const uint32_t* __restrict__ sm) {
    constexpr uint32_t MT = (1u << T) - 1u;
    constexpr uint32_t MT1 = (2u << T) - 1u;
    constexpr uint32_t MROW = (4u << T) - 1u;
    constexpr int R = DEAD ? T : T + 1;               // S5: the +y halo row belongs to the (active) tile above
    constexpr int NB = NarrowBatch<T>::N;
    const uint32_t a = x0 >> 5;
    const uint32_t a1 = (a + 1u == W) ? 0u : a + 1u;
    uint32_t g = y0, g2 = y0;
    size_t row = (size_t)y0 * W, row2 = row;
#pragma unroll 1
    for (int r0 = 0; r0 < R; r0 += NB) {
        uint32_t yl[NB], yh[NB], xl[NB], xh[NB];
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            if (r0 + b < R) {
                yl[b] = planeY[row + a];
                yh[b] = planeY[row + a1];
                if (r0 + b < T) {
                    xl[b] = planeX[row + a];
                    xh[b] = planeX[row + a1];
                }
                row += W;
                if (++g == L) { g = 0u; row = 0; }
            }
        }
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const int r = r0 + b;
            if (r < R) {
                const uint32_t ly = (uint32_t)r;
                const uint32_t word = sm[(ly + 1u) * NTHR] ^ (enc_narrow(ly) & MROW);
                const uint32_t below = sm[ly * NTHR] ^ (enc_narrow(ly - 1u) & MROW);
                const uint32_t sy = ((word ^ below) >> 1) ^ ycode(ly);
                store_bits_pre(planeY + row2 + a, planeY + row2 + a1, x0, MT, sy, yl[b], yh[b]);
                if (r < T) {
                    const uint32_t sx = ((word ^ (word << 1)) >> 1) ^ ycode(ly);   // bit lx = h1(lx)^h1(lx-1)^h0(lx,ly), lx = 0..T
                    store_bits_pre(planeX + row2 + a, planeX + row2 + a1, x0, DEAD ? MT : MT1, sx, xl[b], xh[b]);   // S5: bit T belongs to the right tile
                }
                row2 += W;
                if (++g2 == L) { g2 = 0u; row2 = 0; }
            }
        }
    }
}

// ---- a4: one attempt (eq. 2).  MODE 0: p = 1, q = 0 (accept words are never needed and their Philox calls are
// never evaluated -- bit-identical, the generator is counter-based).  MODE 1: p, q both > 0.  MODE 2: any p, q.  TRACK: this
// thread's tile holds global site (0,0) at local index origin_idx.  A flip is one shared-memory XOR reduction
// (ATOMS.XOR without return) with a zero mask when nothing flips: no branch on the outcome, so a whole batch of
// attempts stays one basic block for the instruction scheduler.
__device__ __forceinline__ uint32_t lop3_and_not_not(uint32_t m, uint32_t x, uint32_t y) {
    uint32_t r;   // m & ~x & ~y
    asm("lop3.b32 %0, %1, %2, %3, 0x10;" : "=r"(r) : "r"(m), "r"(x), "r"(y));
    return r;
}

template <int LUT>
__device__ __forceinline__ uint32_t lop3(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t r;   // bitwise function of (a, b, c) with truth table LUT (a = 0xF0, b = 0xCC, c = 0xAA)
    asm("lop3.b32 %0, %1, %2, %3, %4;" : "=r"(r) : "r"(a), "r"(b), "r"(c), "n"(LUT));
    return r;
}

template <int T, int NTHR, int MODE, bool TRACK, bool DEAD>
__device__ __forceinline__ void attempt(uint32_t* __restrict__ sm, uint32_t site_word, uint32_t accept_word,
                                        const UpdateParams& P, uint32_t& n_dep, float& dep_f, uint32_t& n_rem,
                                        float& rem_f, int32_t& dh00, uint32_t origin_idx, bool live = true) {
    using G = TileGeom<T>;
    const uint32_t idx = site_word >> (32 - 2 * G::LOG2T);      // mulhi32(site_word, T*T) = ly*T + lx
    const uint32_t ly = idx >> G::LOG2T;
    uint32_t* a;
    uint32_t wo, wl, wr, sh;
    if constexpr (G::WIDE) {
        // word (row ly+1, k = lx>>5) = PAD + (ly+1)*WPR + k, and idx>>5 = ly*WPL + k
        a = sm + ((idx >> 5) + ly + (uint32_t)(G::PAD + G::WPR)) * NTHR;
        wo = a[0];
        const uint32_t wp = *(a - NTHR), wn = a[NTHR];
        wl = __funnelshift_l(wp, wo, 1);      // left neighbours aligned with their site
        wr = __funnelshift_r(wo, wn, 1);      // right neighbours
        sh = idx;                             // low 5 bits = lx & 31
    } else {
        a = sm + (ly + 1u) * NTHR;
        wo = a[0];
        wl = wo << 1;
        wr = wo >> 1;
        sh = (idx & (uint32_t)(T - 1)) + 1u;
    }
    const uint32_t wd = *(a - G::WPR * NTHR), wu = a[G::WPR * NTHR];
    uint32_t bit = __funnelshift_l(0u, 1u, sh);                 // 1 << (sh & 31)
    if (DEAD) {
        // dead-border schedule S5: an attempt on the +x or +y edge of the tile does nothing
        const bool edge = (((idx + 1u) & (uint32_t)(T - 1)) == 0u) || (idx >= (uint32_t)(T * (T - 1)));
        bit = edge ? 0u : bit;
    }
    bit = live ? bit : 0u;      // S7: steps beyond the tile's Poissonised count (constant true elsewhere)
    // parity-free encoding (enc_word / enc_narrow): minimum <=> right, up equal the site's bit and left, down differ;
    // t1, t2 (u1, u2): set where the site is NOT a minimum (maximum) along x, y
    const uint32_t t1 = lop3<0xDB>(wo, wl, wr);      // (o^~l)|(o^r)
    const uint32_t t2 = lop3<0xBD>(wo, wu, wd);      // (o^u)|(o^~d)
    uint32_t u1 = 0u, u2 = 0u;
    if (MODE != 0) {
        u1 = lop3<0xBD>(wo, wl, wr);
        u2 = lop3<0xDB>(wo, wu, wd);
    }
    if (MODE == 0) {
        const uint32_t md0 = lop3_and_not_not(bit, t1, t2);
        atomicXor(a, md0);
        // deposits of this tile counted in fp32 (exact: at most T*T < 2^24 per tile and launch): the predicated
        // FADD runs on the FMA pipe, the integer pipe is the busy one
        asm("{ .reg .pred p; setp.ne.u32 p, %1, 0; @p add.f32 %0, %0, 0f3F800000; }" : "+f"(dep_f) : "r"(md0));
        if (TRACK) dh00 += (md0 != 0u && idx == origin_idx) ? 2 : 0;
    } else if (MODE == 1) {
        // both probabilities > 0: 32-bit inclusive thresholds.  The two accept decisions do not depend on the
        // lattice, so they are taken off the dependent chain (loads -> tests -> XOR): the site bit is masked by
        // each decision beforehand.  A site is never a minimum and a maximum at once: md and mr are disjoint.
        const uint32_t bit_p = (accept_word <= P.tp_incl) ? bit : 0u;
        const uint32_t bit_q = (accept_word <= P.tq_incl) ? bit : 0u;
        const uint32_t md = lop3_and_not_not(bit_p, t1, t2);
        const uint32_t mr = lop3_and_not_not(bit_q, u1, u2);
        atomicXor(a, md | mr);
        asm("{ .reg .pred p; setp.ne.u32 p, %1, 0; @p add.f32 %0, %0, 0f3F800000; }" : "+f"(dep_f) : "r"(md));
        asm("{ .reg .pred p; setp.ne.u32 p, %1, 0; @p add.f32 %0, %0, 0f3F800000; }" : "+f"(rem_f) : "r"(mr));
        if (TRACK) dh00 += (idx == origin_idx) ? (md ? 2 : (mr ? -2 : 0)) : 0;
    } else {
        // general thresholds (a probability of exactly 0 with the other one in (0,1])
        const uint32_t md = ((uint64_t)accept_word < P.thr_p) ? lop3_and_not_not(bit, t1, t2) : 0u;
        const uint32_t mr = ((uint64_t)accept_word < P.thr_q) ? lop3_and_not_not(bit, u1, u2) : 0u;
        atomicXor(a, md | mr);
        n_dep += (md != 0u) ? 1u : 0u;
        n_rem += (mr != 0u) ? 1u : 0u;
        if (TRACK) dh00 += (idx == origin_idx) ? (md ? 2 : (mr ? -2 : 0)) : 0;
    }
}


// T*T sequential attempts of one tile (S3).  Site call c serves steps 8c..8c+7: each of its four words is a
// base-T*T fraction with two digits (for the power-of-two T*T of this path: its top 2*log2(T) bits and the next
// 2*log2(T) bits).  Accept calls 2c and 2c+1 (counter | 2^31) serve the same eight steps, one word each, and are
// evaluated only in MODE 1.  Calls are generated one batch ahead of the attempts that consume them (the generator
// is counter-based, so the next batch does not depend on the lattice): the multiplier pipe works on batch b+1
// while the shared-memory round trips of batch b are in flight.
template <int T, int NTHR, int MODE, bool TRACK, bool DEAD, int SUBM>
__device__ __forceinline__ void run_tile_steps(uint32_t* __restrict__ sm, const UpdateParams& P, uint32_t tile_id,
                                               uint32_t replica, uint32_t& n_dep, uint32_t& n_rem, int32_t& dh00,
                                               uint32_t origin_idx, uint32_t n_steps) {
    constexpr bool WHOLE = (SUBM == 0);
    constexpr uint32_t ACCEPT = 0x80000000u;
    constexpr uint32_t TT = (uint32_t)(T * T);
    // WHOLE: all T*T/8 site calls of the tile (compile-time trip count); otherwise one sub-sweep's slice (S6)
    // SUBM 2 (S7): the sub-sweep's own stream region (steps from sub * 2^16), n_steps of them for this tile
    const uint32_t c_begin = WHOLE ? 0u : (SUBM == 2 ? (P.sub << 13) : P.call_begin);
    const uint32_t c_end = WHOLE ? (uint32_t)(T * T) / 8u : (SUBM == 2 ? c_begin + ((n_steps + 7u) >> 3) : P.call_end);
    uint4 cur, nxt, cur_a[2], nxt_a[2];
    float dep_f = 0.0f, rem_f = 0.0f;       // MODE 0, 1: deposits / removals of this tile (see attempt)
    cur = philox4x32_10(c_begin, tile_id, P.m, replica, P.key);
    if (MODE) {
        cur_a[0] = philox4x32_10((2u * c_begin) | ACCEPT, tile_id, P.m, replica, P.key);
        cur_a[1] = philox4x32_10((2u * c_begin + 1u) | ACCEPT, tile_id, P.m, replica, P.key);
    }
    // measured on B200 at L = 2^16: 4 calls (32 attempts) per loop body are 4.5 % faster than 1 with the accept
    // stream off, 2 are best with it on; 16 overflow the instruction cache
    constexpr int UNROLL = (MODE == 0) ? 4 : 2;
#pragma unroll UNROLL
    for (uint32_t c = c_begin; c < c_end; ++c) {
        // batch c+1 (the last iteration generates one unused batch)
        nxt = philox4x32_10(c + 1u, tile_id, P.m, replica, P.key);
        if (MODE) {
            nxt_a[0] = philox4x32_10((2u * c + 2u) | ACCEPT, tile_id, P.m, replica, P.key);
            nxt_a[1] = philox4x32_10((2u * c + 3u) | ACCEPT, tile_id, P.m, replica, P.key);
        }
        const uint32_t rem = n_steps - 8u * (c - c_begin);      // S7: live steps left in this call and after
        const uint4 a0 = MODE ? cur_a[0] : make_uint4(0u, 0u, 0u, 0u);
        const uint4 a1 = MODE ? cur_a[1] : make_uint4(0u, 0u, 0u, 0u);
        attempt<T, NTHR, MODE, TRACK, DEAD>(sm, cur.x, a0.x, P, n_dep, dep_f, n_rem, rem_f, dh00, origin_idx, SUBM != 2 || rem > 0u);
        attempt<T, NTHR, MODE, TRACK, DEAD>(sm, cur.x * TT, a0.y, P, n_dep, dep_f, n_rem, rem_f, dh00, origin_idx, SUBM != 2 || rem > 1u);
        attempt<T, NTHR, MODE, TRACK, DEAD>(sm, cur.y, a0.z, P, n_dep, dep_f, n_rem, rem_f, dh00, origin_idx, SUBM != 2 || rem > 2u);
        attempt<T, NTHR, MODE, TRACK, DEAD>(sm, cur.y * TT, a0.w, P, n_dep, dep_f, n_rem, rem_f, dh00, origin_idx, SUBM != 2 || rem > 3u);
        attempt<T, NTHR, MODE, TRACK, DEAD>(sm, cur.z, a1.x, P, n_dep, dep_f, n_rem, rem_f, dh00, origin_idx, SUBM != 2 || rem > 4u);
        attempt<T, NTHR, MODE, TRACK, DEAD>(sm, cur.z * TT, a1.y, P, n_dep, dep_f, n_rem, rem_f, dh00, origin_idx, SUBM != 2 || rem > 5u);
        attempt<T, NTHR, MODE, TRACK, DEAD>(sm, cur.w, a1.z, P, n_dep, dep_f, n_rem, rem_f, dh00, origin_idx, SUBM != 2 || rem > 6u);
        attempt<T, NTHR, MODE, TRACK, DEAD>(sm, cur.w * TT, a1.w, P, n_dep, dep_f, n_rem, rem_f, dh00, origin_idx, SUBM != 2 || rem > 7u);
        cur = nxt;
        if (MODE) {
            cur_a[0] = nxt_a[0];
            cur_a[1] = nxt_a[1];
        }
    }
    n_dep += (uint32_t)dep_f;
    n_rem += (uint32_t)rem_f;
}

// DEAD = false: one colour of schedule S4 per launch (P.slot);  DEAD = true: every tile of the dead-border schedule
// S5 in one launch (P.HN = NT).
// SUB = 1: one sub-sweep (S6), site calls [P.call_begin, P.call_end) of every tile instead of all of them.
// SUB = 2: Poissonised number of steps per tile (S7), drawn here from the count call and the table P.pthr.
template <int T, int NTHR, int MODE, bool DEAD, int SUB>
// T = 64: CTAs of 96 threads, three per SM = 9 warps (eight 32-thread CTAs are the limit otherwise: 1 KB of shared
// memory is reserved per CTA); measured on B200 at L = 2^16: 690 against 681 Gupd/s
// T = 32: 64-thread CTAs; asking for 8 per SM caps the registers at 125 (16 warps per SM: 834 against 790 Gupd/s at
// L = 2^16; tighter caps spill and slow the small, chain-bound lattices of config 2)
__global__ void __launch_bounds__(NTHR, (T == 64) ? 3 : (T == 32 ? 8 : 1)) kpz_update_kernel(const UpdateParams P) {
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
    global_draw<T>(P, SUB ? P.sub : 0u, replica, ox, oy, colour);
    const uint32_t tx = DEAD ? i : 2u * i + (colour & 1u);
    uint32_t tyl = DEAD ? j : 2u * (j + P.j0) + (colour >> 1);
    if (tyl >= P.tywrap) tyl -= P.tywrap;                     // a launch over a wrapped range of tile rows
    const uint32_t ty = tyl + P.ty0;                          // global tile row (tyl: within the stored rows)
    const uint32_t X0 = ox + tx * T, Y0 = oy + tyl * T;       // < L + T
    const uint32_t tile_id = ty * P.NT + tx;
    uint32_t* planeX = P.lattice + (size_t)replica * 2u * P.plane_words;
    uint32_t* planeY = planeX + P.plane_words;
    const uint32_t L = P.L, W = P.W, LY = P.ywrap;
    const uint32_t x0 = (X0 >= L) ? X0 - L : X0;   // first own column = bit offset inside a row
    const uint32_t y0 = (Y0 >= LY) ? Y0 - LY : Y0; // first own row (storage index)
    const uint32_t Yg = oy + ty * T;               // ... and as a global row, for the origin test
    const uint32_t yg0 = (Yg >= L) ? Yg - L : Yg;

    uint32_t n_dep = 0, n_rem = 0, n_att = 0;
    int32_t dh00 = 0;
    uint32_t origin_idx = 0xFFFFFFFFu;
    if (active) {
        // ---- a2: stage tile + halo ----
        if constexpr (G::WIDE) stage_in_wide<T, NTHR>(planeX, planeY, LY, W, x0, y0, sm);
        else stage_in_narrow<T, NTHR>(planeX, planeY, LY, W, x0, y0, sm);
        // does this tile hold global site (0,0)?  its local coordinates: (L - x0) mod L, (L - yg0) mod L
        const uint32_t lx0 = (x0 == 0u) ? 0u : L - x0;
        const uint32_t ly0 = (yg0 == 0u) ? 0u : L - yg0;
        if (lx0 < (uint32_t)T && ly0 < (uint32_t)T) origin_idx = ly0 * T + lx0;
    }
    const bool any_origin = __any_sync(0xFFFFFFFFu, origin_idx != 0xFFFFFFFFu);
    if (active) {
        // ---- a3 + a4: T*T sequential attempts ----
        uint32_t n_steps = 0u;
        if (SUB == 2) {
            // n = pk_min + #{i < pn - 1 : pthr[i] <= u}: upper bound in the monotone table
            const uint32_t u = philox4x32_10(0x7FFFFFFFu - P.sub, tile_id, P.m, replica, P.key).x;
            uint32_t lo = 0u, hi = P.pn - 1u;
            while (lo < hi) {
                const uint32_t mid = (lo + hi) >> 1;
                if (P.pthr[mid] <= (unsigned long long)u) lo = mid + 1u; else hi = mid;
            }
            n_steps = P.pk_min + lo;
            n_att = n_steps;
        }
        if (any_origin)
            run_tile_steps<T, NTHR, MODE, true, DEAD, SUB>(sm, P, tile_id, replica, n_dep, n_rem, dh00, origin_idx, n_steps);
        else
            run_tile_steps<T, NTHR, MODE, false, DEAD, SUB>(sm, P, tile_id, replica, n_dep, n_rem, dh00, origin_idx, n_steps);
        // ---- a5: write back ----
        if constexpr (G::WIDE) stage_out_wide<T, NTHR, StageBatch<T>::N, DEAD>(planeX, planeY, LY, W, x0, y0, sm);
        else stage_out_narrow<T, NTHR, DEAD>(planeX, planeY, LY, W, x0, y0, sm);
    }
    // ---- a6: bookkeeping ----
    const uint32_t rep0 = __shfl_sync(0xFFFFFFFFu, replica, 0);
    const bool uniform = __all_sync(0xFFFFFFFFu, replica == rep0 && active);
    if (uniform) {
        uint32_t d = n_dep, r = n_rem, a = n_att;
        int32_t h = dh00;
#pragma unroll
        for (int sft = 16; sft > 0; sft >>= 1) {
            d += __shfl_xor_sync(0xFFFFFFFFu, d, sft);
            r += __shfl_xor_sync(0xFFFFFFFFu, r, sft);
            h += __shfl_xor_sync(0xFFFFFFFFu, h, sft);
            if (SUB == 2) a += __shfl_xor_sync(0xFFFFFFFFu, a, sft);
        }
        if ((threadIdx.x & 31u) == 0u) {
            unsigned long long* st = P.stats + (size_t)rep0 * 4u;
            if (d) atomicAdd(st + 0, (unsigned long long)d);
            if (r) atomicAdd(st + 1, (unsigned long long)r);
            if (h) atomicAdd(st + 2, (unsigned long long)(long long)h);
            if (SUB == 2 && a) atomicAdd(st + 3, (unsigned long long)a);
        }
    } else if (active) {
        unsigned long long* st = P.stats + (size_t)replica * 4u;
        if (n_dep) atomicAdd(st + 0, (unsigned long long)n_dep);
        if (n_rem) atomicAdd(st + 1, (unsigned long long)n_rem);
        if (dh00) atomicAdd(st + 2, (unsigned long long)(long long)dh00);
        if (SUB == 2 && n_att) atomicAdd(st + 3, (unsigned long long)n_att);
    }
}


// ------------------------------------------------------------------------------------------------------------
// Lattice-resident variant for small lattices (BASELINE configs 1 and 4: L <= 512).  One CTA copies the packed
// lattices of its G replicas (2 bits per site, the HBM layout) into shared memory ONCE, runs n_mcs whole MCS on
// them -- the four colour passes of an MCS separated by __syncthreads() instead of kernel launches, the global
// draw S2 evaluated in-kernel every pass -- and copies the lattices back.  Every step of a pass is the code of
// kpz_update_kernel itself (stage_in_*, run_tile_steps, stage_out_* with the plane pointers aimed at shared memory),
// so the trajectory is the tiled kernel's bit for bit (schedules S4 and S6); what disappears is the 4 launches per MCS and the global-
// memory round trips of the tile staging, which dominate when a colour has only a few hundred tiles.
// Shared memory: [G][2][L*L/32] lattice words, then TileGeom<T>::WORDS * NTHR words of per-thread tiles.
// STS = true: a flip is written with a plain store of the new word instead of an XOR reduction (the tile words
// are private to their thread); shorter dependent chain, one more integer operation -- for chain-bound launches.
// ------------------------------------------------------------------------------------------------------------
template <int T, int NTHR, int MODE>
__global__ void __launch_bounds__(NTHR) kpz_resident_kernel(const UpdateParams P0, const uint32_t G, const uint32_t n_mcs,
                                                            const uint32_t n_replicas, const uint32_t n_sub) {
    using Geo = TileGeom<T>;
    extern __shared__ uint32_t smem[];
    const uint32_t g0 = blockIdx.x * G;
    const uint32_t ng = min(G, n_replicas - g0);
    const uint32_t lat_words = 2u * (uint32_t)P0.plane_words;          // per replica
    uint32_t* lat = smem;
    uint32_t* sm = smem + G * lat_words + threadIdx.x;
    {
        const uint32_t* src = P0.lattice + (size_t)g0 * lat_words;
        for (uint32_t i = threadIdx.x; i < ng * lat_words; i += NTHR) lat[i] = src[i];
    }
    __syncthreads();
    const uint32_t L = P0.L, W = P0.W;
    const uint32_t items = ng * P0.tiles_per_colour;
    UpdateParams P = P0;
    for (uint32_t mi = 0; mi < n_mcs; ++mi) {
        P.m = P0.m + mi;
        // S6: n_sub sub-sweeps per MCS, each with its own global draw and its slice of every tile's site calls
        // (n_sub = 1: the whole stream, compile-time trip count).  Staging comes from shared memory here, so a
        // sub-sweep costs little more than its attempts.
        for (uint32_t sub = 0; sub < n_sub; ++sub) {
        const uint32_t per = (uint32_t)(T * T / 8) / n_sub;
        P.sub = sub;
        P.call_begin = sub * per;
        P.call_end = (sub + 1u) * per;
        for (uint32_t slot = 0; slot < 4u; ++slot) {
            P.slot = slot;
            for (uint32_t base = 0; base < items; base += NTHR) {
                const uint32_t it = base + threadIdx.x;
                const bool active = it < items;
                const uint32_t g = active ? it / P0.tiles_per_colour : 0u;
                const uint32_t wl = active ? it - g * P0.tiles_per_colour : 0u;
                const uint32_t replica = g0 + g;
                const uint32_t j = wl / P0.HN, i = wl - j * P0.HN;
                uint32_t ox, oy, colour;
                global_draw<T>(P, sub, replica, ox, oy, colour);
                const uint32_t tx = 2u * i + (colour & 1u), ty = 2u * j + (colour >> 1);
                const uint32_t X0 = ox + tx * T, Y0 = oy + ty * T;
                const uint32_t tile_id = ty * P0.NT + tx;
                uint32_t* planeX = lat + g * lat_words;
                uint32_t* planeY = planeX + (uint32_t)P0.plane_words;
                const uint32_t x0 = (X0 >= L) ? X0 - L : X0;
                const uint32_t y0 = (Y0 >= L) ? Y0 - L : Y0;
                uint32_t n_dep = 0, n_rem = 0;
                int32_t dh00 = 0;
                uint32_t origin_idx = 0xFFFFFFFFu;
                if (active) {
                    if constexpr (Geo::WIDE) stage_in_wide<T, NTHR>(planeX, planeY, L, W, x0, y0, sm);
                    else stage_in_narrow<T, NTHR>(planeX, planeY, L, W, x0, y0, sm);
                    const uint32_t lx0 = (x0 == 0u) ? 0u : L - x0;
                    const uint32_t ly0 = (y0 == 0u) ? 0u : L - y0;
                    if (lx0 < (uint32_t)T && ly0 < (uint32_t)T) origin_idx = ly0 * T + lx0;
                }
                const bool any_origin = __any_sync(0xFFFFFFFFu, origin_idx != 0xFFFFFFFFu);
                if (active) {
                    if (n_sub == 1u) {
                        if (any_origin)
                            run_tile_steps<T, NTHR, MODE, true, false, 0>(sm, P, tile_id, replica, n_dep, n_rem, dh00, origin_idx, 0u);
                        else
                            run_tile_steps<T, NTHR, MODE, false, false, 0>(sm, P, tile_id, replica, n_dep, n_rem, dh00, origin_idx, 0u);
                    } else {
                        // TRACK = true is correct for every tile (it only adds the origin test): one instance less
                        run_tile_steps<T, NTHR, MODE, true, false, 1>(sm, P, tile_id, replica, n_dep, n_rem, dh00, origin_idx, 0u);
                    }
                    if constexpr (Geo::WIDE) stage_out_wide<T, NTHR, StageBatch<T>::N, false>(planeX, planeY, L, W, x0, y0, sm);
                    else stage_out_narrow<T, NTHR, false>(planeX, planeY, L, W, x0, y0, sm);
                    unsigned long long* st = P0.stats + (size_t)replica * 4u;
                    if (n_dep) atomicAdd(st + 0, (unsigned long long)n_dep);
                    if (n_rem) atomicAdd(st + 1, (unsigned long long)n_rem);
                    if (dh00) atomicAdd(st + 2, (unsigned long long)(long long)dh00);
                }
            }
            __syncthreads();
        }
        }
    }
    {
        uint32_t* dst = P0.lattice + (size_t)g0 * lat_words;
        for (uint32_t i = threadIdx.x; i < ng * lat_words; i += NTHR) dst[i] = lat[i];
    }
}


}  // namespace kpz
