// kpz_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct CPU oracle for the octahedron-KPZ hot path of
// Kelling & Odor, arXiv:1110.6745 (PAPER.md; "P:n" = PAPER.md line n).  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build,
// load or call this file.  It shares no code, header, table or helper with the CUDA path
// (paper_1110_6745_b200/csrc) and neither includes the other.
//
// What it follows, step by step (readings of garbled / silent passages: DESIGN.md "Readings"):
//   * state      : unpacked int8 slopes sx(x,y) = h(x,y)-h(x-1,y), sy(x,y) = h(x,y)-h(x,y-1), values +-1,
//                  periodic L x L (reading R1 "down = -1", R3 backward difference).
//   * rule       : eq. (2).  (sx(x,y), sx(x+1,y); sy(x,y), sy(x,y+1)) = (-1,+1; -1,+1) -> (+1,-1; +1,-1)
//                  with probability p (deposition, h(x,y) += 2); the reverse with probability q.
//   * schedule   : DESIGN.md section "Schedule" (the paper fixes none for the north star): per MCS one global
//                  Philox draw -> offset (ox,oy) multiples of g and an order of the 4 tile colours;
//                  every tile of the active colour performs T*T sequential single-site attempts.
//   * RNG        : Philox4x32-10 (Salmon et al., SC'11), written out below; pinned by the published known answers.
//   * heights    : eq. (3), P:34 (reading R4): h(x,y) = h00 + sum_{l=1..x} sx(l,0) + sum_{k=1..y} sy(x,k).
//   * width      : eq. (4), P:37-40 (reading R5): W2 = (1/N) sum h^2 - ((1/N) sum h)^2, N = L*L.
//
// Parity pins (tests/test_oracle_*.py): Philox KAT, W2(flat) = 1/4, triangle-wave closed form,
// conservation + curl-free after every step, +2 per accepted flip, exact L=4 / L=6 Markov chains.
// "parity unpinned" (definitions of this build, pinned only by the independent Python twin in
// oracle/kpz_twin.py and by distribution tests): tile-colour order decode, offset draw, step -> Philox word map.
// kpzo_state_hash is a checksum, not part of the method, and is "parity unpinned" as well (both sides restate the
// formula of SURVEY 8(b)); no parity case relies on it alone.
//
// Optional OpenMP: tiles of one colour are independent,
// so the tile loop may run in parallel; results are identical for any thread count.  The same holds for the
// loops over rows in kpzo_init_flat, over columns in kpzo_measure and over sites in kpzo_state_hash (exact
// integer sums of independent terms): they are parallel too, so that the full-lattice parity cases at L = 2^16 and
// 2^17 finish in minutes.  No arithmetic differs from the serial loops.

#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

typedef unsigned __int128 u128;
typedef __int128 i128;

// ---- Philox4x32-10, Salmon/Moraes/Dror/Shaw SC'11 (public algorithm), restated ------------------------------
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        if (round > 0) { k0 += W0; k1 += W1; }
        uint64_t p0 = (uint64_t)M0 * c0;
        uint64_t p1 = (uint64_t)M1 * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

inline uint32_t mulhi32(uint32_t a, uint32_t n) { return (uint32_t)(((uint64_t)a * n) >> 32); }

// accept threshold: accept iff (uint64)word < thr ; thr = 2^32 if prob >= 1 else floor(prob * 2^32)
uint64_t threshold(double prob) {
    if (prob >= 1.0) return (uint64_t)1 << 32;
    if (prob <= 0.0) return 0;
    return (uint64_t)(prob * 4294967296.0);   // floor for positive values
}

struct Oracle {
    uint32_t L, T, g, NT;
    uint64_t seed;
    uint32_t replica;
    double p, q;
    uint64_t thr_p, thr_q;
    // window (global coordinates of the stored region); full lattice: wx0 = wy0 = 0, ww = wh = L
    uint32_t wx0, wy0, ww, wh;
    bool full;
    std::vector<int8_t> sx, sy;       // [wy][wx]
    std::vector<int32_t> H;           // shadow heights (only when shadow = true)
    bool shadow;
    int64_t h00;
    uint64_t mcs, attempts, deposits, removals;
    int nthreads;
    uint32_t sub_sweeps;   // K >= 1 sub-sweeps per MCS (S6); K divides T*T
    bool poisson;          // S7: Poissonised number of steps per tile and sub-sweep
    uint32_t pk_min;       // smallest count of the table
    std::vector<uint64_t> pthr;   // pthr[i] = floor(2^32 * P(n <= pk_min + i)), last entry 2^32
    int schedule;      // 0: four tile colours with halo (S4); 1: dead borders, one pass (S5)
};

inline bool in_window(const Oracle* o, uint32_t x, uint32_t y, size_t* idx) {
    uint32_t rx = (x + o->L - o->wx0) % o->L;
    uint32_t ry = (y + o->L - o->wy0) % o->L;
    if (rx >= o->ww || ry >= o->wh) return false;
    *idx = (size_t)ry * o->ww + rx;
    return true;
}

// One single-site attempt at global site (x,y) with accept word a.  eq. (2).
// Returns +1 deposition, -1 removal, 0 nothing.
inline int attempt(Oracle* o, uint32_t x, uint32_t y, uint32_t accept_word) {
    const uint32_t L = o->L;
    size_t i0, ix, iy;
    if (!in_window(o, x, y, &i0)) return 0;
    if (!in_window(o, (x + 1) % L, y, &ix)) return 0;
    if (!in_window(o, x, (y + 1) % L, &iy)) return 0;
    int8_t a = o->sx[i0], b = o->sx[ix], c = o->sy[i0], d = o->sy[iy];
    int dir = 0;
    if (a == -1 && b == +1 && c == -1 && d == +1) {
        if ((uint64_t)accept_word < o->thr_p) dir = +1;
    } else if (a == +1 && b == -1 && c == +1 && d == -1) {
        if ((uint64_t)accept_word < o->thr_q) dir = -1;
    }
    if (dir != 0) {
        o->sx[i0] = (int8_t)-a; o->sx[ix] = (int8_t)-b;
        o->sy[i0] = (int8_t)-c; o->sy[iy] = (int8_t)-d;
        if (o->shadow) o->H[i0] += 2 * dir;
    }
    return dir;
}

// global draw of MCS m: offset and colour order.  DESIGN.md "Schedule" S2.
void global_draw(const Oracle* o, uint32_t m, uint32_t sub, uint32_t* ox, uint32_t* oy, uint32_t perm[4]) {
    uint32_t ctr[4] = {sub, 0xFFFFFFFFu, m, o->replica};   // S6: sub-sweep j of MCS m draws with c0 = j (j = 0: S2)
    uint32_t key[2] = {(uint32_t)(o->seed & 0xFFFFFFFFu), (uint32_t)(o->seed >> 32)};
    uint32_t G[4];
    philox4x32_10(ctr, key, G);
    *ox = o->g * mulhi32(G[0], o->T / o->g);
    *oy = o->g * mulhi32(G[1], o->T / o->g);
    uint32_t pidx = mulhi32(G[2], 24);
    uint32_t d0 = pidx / 6, d1 = (pidx % 6) / 2, d2 = pidx % 2;
    uint32_t pool[4] = {0, 1, 2, 3};
    int n = 4;
    uint32_t digits[3] = {d0, d1, d2};
    for (int k = 0; k < 3; ++k) {
        perm[k] = pool[digits[k]];
        for (int j = (int)digits[k]; j < n - 1; ++j) pool[j] = pool[j + 1];
        --n;
    }
    perm[3] = pool[0];
}

// S7: integer-defined Poisson table for lambda = T*T/K.  Weights q_lambda = 2^52 at the mode, q_k = floor(q_{k-1}
// * lambda / k) above it and q_k = floor(q_{k+1} * (k+1) / lambda) below it, for |k - lambda| <= W =
// ceil(12 sqrt(lambda)) + 16 (k >= 0); thresholds floor(2^32 * C_k / S) with C_k the running sum and S the total.
void build_poisson_table(Oracle* o) {
    const uint64_t lam = (uint64_t)o->T * o->T / o->sub_sweeps;
    uint64_t W = 16;
    while ((W - 16) * (W - 16) < 144 * lam) ++W;              // W - 16 = ceil(12 sqrt(lambda))
    const uint64_t kmin = lam > W ? lam - W : 0, kmax = lam + W;
    std::vector<u128> q(kmax - kmin + 1);
    q[lam - kmin] = (u128)1 << 52;
    for (uint64_t k = lam + 1; k <= kmax; ++k) q[k - kmin] = q[k - 1 - kmin] * lam / k;
    for (uint64_t k = lam; k-- > kmin;) q[k - kmin] = q[k + 1 - kmin] * (k + 1) / lam;
    u128 S = 0;
    for (u128 v : q) S += v;
    o->pk_min = (uint32_t)kmin;
    o->pthr.resize(q.size());
    u128 C = 0;
    for (size_t i = 0; i < q.size(); ++i) {
        C += q[i];
        o->pthr[i] = (uint64_t)((C << 32) / S);
    }
}

// number of steps of tile `tile_id` in sub-sweep `sub` of MCS m: kmin + #{i : pthr[i] <= u}, u = word 0 of the
// count call R(0x7FFFFFFF - sub, tile_id, m, replica)
uint32_t poisson_count(const Oracle* o, uint32_t m, uint32_t sub, uint32_t tile_id) {
    const uint32_t ctr[4] = {0x7FFFFFFFu - sub, tile_id, m, o->replica};
    const uint32_t key[2] = {(uint32_t)(o->seed & 0xFFFFFFFFu), (uint32_t)(o->seed >> 32)};
    uint32_t Q[4];
    philox4x32_10(ctr, key, Q);
    uint32_t n = o->pk_min;
    for (size_t i = 0; i + 1 < o->pthr.size(); ++i)
        if (o->pthr[i] <= (uint64_t)Q[0]) ++n;
    return n;
}

// all T*T sequential steps of tile (tx,ty) in MCS m.  DESIGN.md "Schedule" S3.
void run_tile(Oracle* o, uint32_t m, uint32_t ox, uint32_t oy, uint32_t tx, uint32_t ty,
              uint64_t* n_dep, uint64_t* n_rem, int64_t* dh00, uint32_t s_begin, uint32_t s_end) {
    const uint32_t T = o->T, L = o->L;
    const uint32_t tile_id = ty * o->NT + tx;
    const uint32_t key[2] = {(uint32_t)(o->seed & 0xFFFFFFFFu), (uint32_t)(o->seed >> 32)};
    const uint32_t steps = T * T;
    // S3: a 32-bit site word W is read as a base-T*T fraction and gives two site indices,
    //   digit 0 = mulhi32(W, T*T),  digit 1 = mulhi32((W * T*T) mod 2^32, T*T);
    // step s takes digit s & 1 of word (s >> 1) & 3 of call R(s >> 3, ...); its accept word is word s & 3 of call
    // R((s >> 2) | 0x80000000, ...).
    uint32_t QS[4] = {0, 0, 0, 0}, QA[4] = {0, 0, 0, 0};
    if (o->poisson) {
        // S7: sub-sweep j = s_begin / (T*T/K) owns the stream region starting at step j * 2^16 and runs n steps of it
        const uint32_t sub = s_begin / (steps / o->sub_sweeps);
        s_begin = sub << 16;
        s_end = s_begin + poisson_count(o, m, sub, tile_id);
        #pragma omp atomic
        o->attempts += (uint64_t)(s_end - s_begin);
    }
    for (uint32_t s = s_begin; s < s_end; ++s) {
        if ((s & 7u) == 0u || s == s_begin) {
            uint32_t ctr_s[4] = {s >> 3, tile_id, m, o->replica};
            philox4x32_10(ctr_s, key, QS);
        }
        if ((s & 3u) == 0u || s == s_begin) {
            uint32_t ctr_a[4] = {(s >> 2) | 0x80000000u, tile_id, m, o->replica};
            philox4x32_10(ctr_a, key, QA);
        }
        uint32_t site_word = QS[(s >> 1) & 3u];
        if (s & 1u) site_word = site_word * steps;      // second digit: fractional part of W * T*T
        uint32_t accept_word = QA[s & 3u];
        uint32_t idx = mulhi32(site_word, steps);
        uint32_t lx = idx % T, ly = idx / T;
        // S5: "if a thread hits a site belonging to a block border it does nothing" -- the +x and +y edge
        // sites of a tile are the ones whose update would change slopes stored in the neighbouring tile (Fig. 1)
        if (o->schedule == 1 && (lx == T - 1 || ly == T - 1)) continue;
        uint32_t x = (ox + tx * T + lx) % L;
        uint32_t y = (oy + ty * T + ly) % L;
        int dir = attempt(o, x, y, accept_word);
        if (dir > 0) ++*n_dep;
        if (dir < 0) ++*n_rem;
        if (dir != 0 && x == 0 && y == 0) *dh00 += 2 * dir;
    }
}

bool tile_touches_window(const Oracle* o, uint32_t ox, uint32_t oy, uint32_t tx, uint32_t ty) {
    if (o->full) return true;
    // tile covers x in [sx0, sx0+T) mod L, the window covers [wx0, wx0+ww) mod L: two periodic intervals meet
    // iff the start of one lies inside the other.
    const uint32_t L = o->L, T = o->T;
    const uint32_t sx0 = (ox + tx * T) % L, sy0 = (oy + ty * T) % L;
    const bool hitx = ((sx0 + L - o->wx0) % L < o->ww) || ((o->wx0 + L - sx0) % L < T);
    const bool hity = ((sy0 + L - o->wy0) % L < o->wh) || ((o->wy0 + L - sy0) % L < T);
    return hitx && hity;
}

// one sub-sweep: steps [s_begin, s_end) of every tile's stream of MCS m, in the frame and colour order of draw `sub`
void run_sub_sweep(Oracle* o, uint32_t m, uint32_t sub, uint32_t s_begin, uint32_t s_end) {
    uint32_t ox, oy, perm[4];
    global_draw(o, m, sub, &ox, &oy, perm);
    const uint32_t NT = o->NT;
    if (o->schedule == 1) {
        // S5: every tile in one pass; the tiles are independent because their edge sites are dead
        uint64_t n_dep = 0, n_rem = 0;
        int64_t dh00 = 0;
        #pragma omp parallel for collapse(2) reduction(+ : n_dep, n_rem, dh00) schedule(dynamic, 16) num_threads(o->nthreads)
        for (int64_t ty = 0; ty < (int64_t)NT; ++ty) {
            for (int64_t tx = 0; tx < (int64_t)NT; ++tx) {
                if (!tile_touches_window(o, ox, oy, (uint32_t)tx, (uint32_t)ty)) continue;
                run_tile(o, m, ox, oy, (uint32_t)tx, (uint32_t)ty, &n_dep, &n_rem, &dh00, s_begin, s_end);
            }
        }
        o->deposits += n_dep; o->removals += n_rem; o->h00 += dh00;
        return;
    }
    for (int i = 0; i < 4; ++i) {
        const uint32_t colour = perm[i];
        const uint32_t cx = colour & 1u, cy = colour >> 1;
        uint64_t n_dep = 0, n_rem = 0;
        int64_t dh00 = 0;
        const int64_t half = NT / 2;
        #pragma omp parallel for collapse(2) reduction(+ : n_dep, n_rem, dh00) schedule(dynamic, 16) num_threads(o->nthreads)
        for (int64_t j = 0; j < half; ++j) {
            for (int64_t k = 0; k < half; ++k) {
                uint32_t ty = (uint32_t)(2 * j) + cy, tx = (uint32_t)(2 * k) + cx;
                if (!tile_touches_window(o, ox, oy, tx, ty)) continue;
                run_tile(o, m, ox, oy, tx, ty, &n_dep, &n_rem, &dh00, s_begin, s_end);
            }
        }
        o->deposits += n_dep; o->removals += n_rem; o->h00 += dh00;
    }
}

// S4 / S5 / S6: one MCS = K sub-sweeps, sub-sweep j executing steps [j T^2/K, (j+1) T^2/K) of every tile
void run_one_mcs(Oracle* o) {
    const uint32_t m = (uint32_t)o->mcs;
    const uint32_t steps = o->T * o->T, K = o->sub_sweeps;
    for (uint32_t j = 0; j < K; ++j) run_sub_sweep(o, m, j, j * (steps / K), (j + 1) * (steps / K));
    if (!o->poisson) o->attempts += (uint64_t)o->L * o->L;     // S7 counts the steps it really made (run_tile)
    o->mcs += 1;
}

// full invariant check (full lattice only).  Returns 0 if all hold, else a bit mask of failures:
// 1 = a slope is not +-1, 2 = some row sum of sx != 0 ... (conservation; zero tilt for states reached from flat),
// 4 = some column sum of sy != 0, 8 = curl: sx(x+1,y)+sy(x+1,y+1) != sy(x,y+1)+sx(x+1,y+1),
// 16 = shadow heights disagree with slopes or with h00.
int check_invariants(const Oracle* o, const int64_t* row_sums_ref, const int64_t* col_sums_ref) {
    if (!o->full) return -1;
    const uint32_t L = o->L;
    int bad = 0;
    for (size_t i = 0; i < (size_t)L * L; ++i) {
        if (o->sx[i] != 1 && o->sx[i] != -1) bad |= 1;
        if (o->sy[i] != 1 && o->sy[i] != -1) bad |= 1;
    }
    for (uint32_t y = 0; y < L; ++y) {
        int64_t s = 0;
        for (uint32_t x = 0; x < L; ++x) s += o->sx[(size_t)y * L + x];
        if (s != (row_sums_ref ? row_sums_ref[y] : 0)) bad |= 2;
    }
    for (uint32_t x = 0; x < L; ++x) {
        int64_t s = 0;
        for (uint32_t y = 0; y < L; ++y) s += o->sy[(size_t)y * L + x];
        if (s != (col_sums_ref ? col_sums_ref[x] : 0)) bad |= 4;
    }
    for (uint32_t y = 0; y < L; ++y)
        for (uint32_t x = 0; x < L; ++x) {
            uint32_t x1 = (x + 1) % L, y1 = (y + 1) % L;
            int a = o->sx[(size_t)y * L + x1] + o->sy[(size_t)y1 * L + x1];
            int b = o->sy[(size_t)y1 * L + x] + o->sx[(size_t)y1 * L + x1];
            if (a != b) bad |= 8;
        }
    if (o->shadow) {
        if (o->H[0] != o->h00) bad |= 16;
        for (uint32_t y = 0; y < L; ++y)
            for (uint32_t x = 0; x < L; ++x) {
                uint32_t xm = (x + L - 1) % L, ym = (y + L - 1) % L;
                if (o->H[(size_t)y * L + x] - o->H[(size_t)y * L + xm] != o->sx[(size_t)y * L + x]) bad |= 16;
                if (o->H[(size_t)y * L + x] - o->H[(size_t)ym * L + x] != o->sy[(size_t)y * L + x]) bad |= 16;
            }
    }
    return bad;
}

}  // namespace

extern "C" {

void kpzo_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); }

uint64_t kpzo_threshold(double prob) { return threshold(prob); }

// T >= 1, L a multiple of 2*T.  g = 4 if T % 4 == 0 else 1 ("multiples of four sites").
// window: (wx0, wy0, ww, wh) in global coordinates; ww = wh = 0 means the full lattice.
void* kpzo_create(uint32_t L, double p, double q, uint32_t T, uint64_t seed, uint32_t replica,
                  uint32_t wx0, uint32_t wy0, uint32_t ww, uint32_t wh, int shadow) {
    if (T < 1 || L < 2 * T || L % (2 * T) != 0) return nullptr;
    if (!(p >= 0.0 && p <= 1.0 && q >= 0.0 && q <= 1.0)) return nullptr;
    Oracle* o = new Oracle();
    o->L = L; o->T = T; o->g = (T % 4 == 0) ? 4 : 1; o->NT = L / T;
    o->seed = seed; o->replica = replica; o->p = p; o->q = q;
    o->thr_p = threshold(p); o->thr_q = threshold(q);
    o->schedule = 0;
    o->sub_sweeps = 1;
    o->poisson = false; o->pk_min = 0;
    o->full = (ww == 0 && wh == 0);
    if (o->full) { wx0 = wy0 = 0; ww = wh = L; }
    if (ww > L || wh > L) { delete o; return nullptr; }
    o->wx0 = wx0 % L; o->wy0 = wy0 % L; o->ww = ww; o->wh = wh;
    o->sx.assign((size_t)ww * wh, 0); o->sy.assign((size_t)ww * wh, 0);
    o->shadow = shadow != 0;
    if (o->shadow) o->H.assign((size_t)ww * wh, 0);
    o->h00 = 0; o->mcs = 0; o->attempts = o->deposits = o->removals = 0;
    o->nthreads = 1;
    return o;
}

void kpzo_destroy(void* h) { delete (Oracle*)h; }

void kpzo_set_threads(void* h, int n) {
    Oracle* o = (Oracle*)h;
#ifdef _OPENMP
    o->nthreads = n > 0 ? n : omp_get_max_threads();
#else
    (void)n; o->nthreads = 1;
#endif
}
int kpzo_get_threads(void* h) { return ((Oracle*)h)->nthreads; }

// flat zig-zag start: h(x,y) = (x+y) mod 2 (W2 = 1/4; reading R7) => sx = sy = +1 if (x+y) odd else -1.
void kpzo_init_flat(void* h) {
    Oracle* o = (Oracle*)h;
    // rows are independent: the loop over ry may run in parallel (plumbing only, same values)
    #pragma omp parallel for schedule(static) num_threads(o->nthreads)
    for (int64_t ry = 0; ry < (int64_t)o->wh; ++ry)
        for (uint32_t rx = 0; rx < o->ww; ++rx) {
            uint32_t x = (o->wx0 + rx) % o->L, y = (o->wy0 + (uint32_t)ry) % o->L;
            int8_t v = ((x + y) & 1u) ? +1 : -1;
            o->sx[(size_t)ry * o->ww + rx] = v;
            o->sy[(size_t)ry * o->ww + rx] = v;
            if (o->shadow) o->H[(size_t)ry * o->ww + rx] = (int32_t)((x + y) & 1u);
        }
    o->h00 = 0; o->mcs = 0; o->attempts = o->deposits = o->removals = 0;
}

// 0 = four tile colours (default), 1 = dead borders.  Returns 0, or -1 for an unknown value.
int kpzo_set_schedule(void* h, int schedule) {
    if (schedule != 0 && schedule != 1) return -1;
    static_cast<Oracle*>(h)->schedule = schedule;
    return 0;
}

// K sub-sweeps per MCS (S6); K >= 1 must divide T*T.  Returns 0 or -1.
int kpzo_set_sub_sweeps(void* h, uint32_t K) {
    Oracle* o = static_cast<Oracle*>(h);
    if (K < 1 || (o->T * o->T) % K != 0) return -1;
    o->sub_sweeps = K;
    if (o->poisson) build_poisson_table(o);
    return 0;
}

// S7 on / off.  Needs T*T/K + W < 2^16 (one stream region per sub-sweep).  Returns 0 or -1.
int kpzo_set_poisson(void* h, int on) {
    Oracle* o = static_cast<Oracle*>(h);
    if (on && (uint64_t)o->T * o->T / o->sub_sweeps > 60000) return -1;
    o->poisson = on != 0;
    if (o->poisson) build_poisson_table(o);
    return 0;
}

// table access for the tests: returns the number of entries, fills kmin and (if thr != NULL) the thresholds
uint32_t kpzo_poisson_table(void* h, uint32_t* kmin, uint64_t* thr) {
    Oracle* o = static_cast<Oracle*>(h);
    if (kmin) *kmin = o->pk_min;
    if (thr) for (size_t i = 0; i < o->pthr.size(); ++i) thr[i] = o->pthr[i];
    return (uint32_t)o->pthr.size();
}

int kpzo_run(void* h, uint64_t n_mcs) {
    Oracle* o = (Oracle*)h;
    for (uint64_t i = 0; i < n_mcs; ++i) {
        if (o->mcs >= 0xFFFFFFFFull) return -1;     // the clock is a 32-bit counter word; 2^32 - 1 MCS at most
        run_one_mcs(o);
    }
    return 0;
}

// Runs n_mcs MCS serially with the full invariant check after EVERY single-site attempt (tiny L only).
// Returns the OR of all failure masks (0 = every invariant held after every step), or -1 if windowed.
// Also checks "+2 per accepted flip": sum of shadow heights changes by exactly 2*dir per step.
int kpzo_run_checked(void* h, uint64_t n_mcs) {
    Oracle* o = (Oracle*)h;
    if (!o->full || !o->shadow) return -1;
    const uint32_t L = o->L, T = o->T;
    std::vector<int64_t> rows(L), cols(L);
    for (uint32_t y = 0; y < L; ++y) { int64_t s = 0; for (uint32_t x = 0; x < L; ++x) s += o->sx[(size_t)y * L + x]; rows[y] = s; }
    for (uint32_t x = 0; x < L; ++x) { int64_t s = 0; for (uint32_t y = 0; y < L; ++y) s += o->sy[(size_t)y * L + x]; cols[x] = s; }
    int bad = check_invariants(o, rows.data(), cols.data());
    const uint32_t key[2] = {(uint32_t)(o->seed & 0xFFFFFFFFu), (uint32_t)(o->seed >> 32)};
    for (uint64_t it = 0; it < n_mcs; ++it) {
        const uint32_t m = (uint32_t)o->mcs;
        uint32_t ox, oy, perm[4];
        global_draw(o, m, 0u, &ox, &oy, perm);
        for (int i = 0; i < 4; ++i) {
            uint32_t cx = perm[i] & 1u, cy = perm[i] >> 1;
            for (uint32_t ty = cy; ty < o->NT; ty += 2)
                for (uint32_t tx = cx; tx < o->NT; tx += 2) {
                    for (uint32_t s = 0; s < T * T; ++s) {
                        uint32_t QS[4], QA[4];
                        uint32_t ctr_s[4] = {s >> 3, ty * o->NT + tx, m, o->replica};
                        uint32_t ctr_a[4] = {(s >> 2) | 0x80000000u, ty * o->NT + tx, m, o->replica};
                        philox4x32_10(ctr_s, key, QS);
                        philox4x32_10(ctr_a, key, QA);
                        uint32_t site_word = QS[(s >> 1) & 3u];
                        if (s & 1u) site_word = site_word * (T * T);
                        uint32_t idx = mulhi32(site_word, T * T);
                        uint32_t x = (ox + tx * T + idx % T) % L, y = (oy + ty * T + idx / T) % L;
                        int64_t before = 0; for (size_t k = 0; k < (size_t)L * L; ++k) before += o->H[k];
                        int dir = attempt(o, x, y, QA[s & 3u]);
                        int64_t after = 0; for (size_t k = 0; k < (size_t)L * L; ++k) after += o->H[k];
                        if (after - before != 2 * dir) bad |= 32;
                        if (dir > 0) o->deposits++;
                        if (dir < 0) o->removals++;
                        if (dir != 0 && x == 0 && y == 0) o->h00 += 2 * dir;
                        bad |= check_invariants(o, rows.data(), cols.data());
                    }
                }
        }
        o->attempts += (uint64_t)L * L;
        o->mcs += 1;
    }
    return bad;
}

int kpzo_check(void* h) { return check_invariants((Oracle*)h, nullptr, nullptr); }

// eq. (3)-(4).  Outputs: sum_h, sum_h2 as 128-bit (lo, hi) pairs of uint64 (two's complement), W2 as double.
// W2 = (N*S2 - S1^2) / N^2: integer numerator (128 bit), one conversion to double, one division by (double)N^2.
int kpzo_measure(void* h, uint64_t* sum_h_lohi, uint64_t* sum_h2_lohi, double* W2) {
    Oracle* o = (Oracle*)h;
    if (!o->full) return -1;
    const uint32_t L = o->L;
    i128 S1 = 0, S2 = 0;
    // walk along x on row 0 from the anchor h(0,0): h(x,0) = h(x-1,0) + sx(x,0)
    std::vector<int64_t> row0(L);
    int64_t hx0 = o->h00;
    for (uint32_t x = 0; x < L; ++x) {
        if (x > 0) hx0 += o->sx[(size_t)0 * L + x];
        row0[x] = hx0;
    }
    // then along y in every column x.  The columns are independent and the sums are exact integers, so the
    // column loop may run in parallel (plumbing only: the same additions in another order).
    #pragma omp parallel num_threads(o->nthreads)
    {
        i128 s1 = 0, s2 = 0;
        #pragma omp for schedule(static) nowait
        for (int64_t x = 0; x < (int64_t)L; ++x) {
            int64_t hh = row0[(size_t)x];
            for (uint32_t y = 0; y < L; ++y) {
                if (y > 0) hh += o->sy[(size_t)y * L + (size_t)x];   // h(x,y) = h(x,y-1) + sy(x,y)
                s1 += hh;
                s2 += (i128)hh * hh;
            }
        }
        #pragma omp critical
        { S1 += s1; S2 += s2; }
    }
    u128 N = (u128)L * L;
    i128 num = (i128)N * S2 - S1 * S1;
    double Nd = (double)((uint64_t)L * L);
    *W2 = (double)num / (Nd * Nd);
    sum_h_lohi[0] = (uint64_t)(u128)S1;  sum_h_lohi[1] = (uint64_t)((u128)S1 >> 64);
    sum_h2_lohi[0] = (uint64_t)(u128)S2; sum_h2_lohi[1] = (uint64_t)((u128)S2 >> 64);
    return 0;
}

// heights by eq. (3) into out[y*L+x] (int32), full lattice
int kpzo_heights(void* h, int32_t* out) {
    Oracle* o = (Oracle*)h;
    if (!o->full) return -1;
    const uint32_t L = o->L;
    int64_t hx0 = o->h00;
    for (uint32_t x = 0; x < L; ++x) {
        if (x > 0) hx0 += o->sx[x];
        int64_t hh = hx0;
        for (uint32_t y = 0; y < L; ++y) {
            if (y > 0) hh += o->sy[(size_t)y * L + x];
            out[(size_t)y * L + x] = (int32_t)hh;
        }
    }
    return 0;
}

// slopes of the stored window, row-major [wh][ww]
void kpzo_get_slopes(void* h, int8_t* sx, int8_t* sy) {
    Oracle* o = (Oracle*)h;
    memcpy(sx, o->sx.data(), o->sx.size());
    memcpy(sy, o->sy.data(), o->sy.size());
}
// sets slopes (values must be +-1); h00 is given; shadow heights rebuilt by eq. (3) (full lattice only)
int kpzo_set_slopes(void* h, const int8_t* sx, const int8_t* sy, int64_t h00) {
    Oracle* o = (Oracle*)h;
    for (size_t i = 0; i < o->sx.size(); ++i)
        if ((sx[i] != 1 && sx[i] != -1) || (sy[i] != 1 && sy[i] != -1)) return -1;
    memcpy(o->sx.data(), sx, o->sx.size());
    memcpy(o->sy.data(), sy, o->sy.size());
    o->h00 = h00;
    if (o->shadow && o->full) kpzo_heights(h, o->H.data());
    return 0;
}
void kpzo_get_shadow(void* h, int32_t* out) {
    Oracle* o = (Oracle*)h;
    if (o->shadow) memcpy(out, o->H.data(), o->H.size() * sizeof(int32_t));
}

void kpzo_counters(void* h, uint64_t* attempts, uint64_t* deposits, uint64_t* removals, int64_t* h00, uint64_t* mcs) {
    Oracle* o = (Oracle*)h;
    *attempts = o->attempts; *deposits = o->deposits; *removals = o->removals; *h00 = o->h00; *mcs = o->mcs;
}

// Sets the MCS clock (Philox counter word c2 of the next MCS, S1) without touching the lattice: the
// state is then "as if" mcs fixed-count MCS had been run (attempts = mcs * L*L).  For parity cases that start a
// trajectory near the end of the 32-bit clock.  Returns 0, or -1 if mcs > 2^32 - 1.
int kpzo_set_clock(void* h, uint64_t mcs) {
    Oracle* o = (Oracle*)h;
    if (mcs > 0xFFFFFFFFull) return -1;
    o->mcs = mcs;
    o->attempts = mcs * (uint64_t)o->L * o->L;
    return 0;
}

void kpzo_global_draw(void* h, uint32_t m, uint32_t* ox, uint32_t* oy, uint32_t* perm) {
    global_draw((Oracle*)h, m, 0u, ox, oy, perm);
}

// True single-site random-sequential reference dynamics (NOT the schedule; used only to bound the bias of the
// domain decomposition, north star "within 3 sigma").  One MCS = L*L attempts at uniformly random sites.
// Stream: Philox counter (attempt_pair_lo, 0xFFFFFFFE, attempt_pair_hi, replica): words (x,y,accept,unused) x 1
// site per call -- its own stream, unrelated to the schedule's.
int kpzo_run_rs(void* h, uint64_t n_mcs) {
    Oracle* o = (Oracle*)h;
    if (!o->full) return -1;
    const uint32_t key[2] = {(uint32_t)(o->seed & 0xFFFFFFFFu), (uint32_t)(o->seed >> 32)};
    const uint64_t per = (uint64_t)o->L * o->L;
    for (uint64_t it = 0; it < n_mcs; ++it) {
        for (uint64_t a = 0; a < per; ++a) {
            uint64_t n = o->attempts + a;
            uint32_t ctr[4] = {(uint32_t)n, 0xFFFFFFFEu, (uint32_t)(n >> 32), o->replica};
            uint32_t Q[4];
            philox4x32_10(ctr, key, Q);
            uint32_t x = mulhi32(Q[0], o->L), y = mulhi32(Q[1], o->L);
            int dir = attempt(o, x, y, Q[2]);
            if (dir > 0) o->deposits++;
            if (dir < 0) o->removals++;
            if (dir != 0 && x == 0 && y == 0) o->h00 += 2 * dir;
        }
        o->attempts += per;
        o->mcs += 1;
    }
    return 0;
}

// order-independent 64-bit state hash: sum over sites of bx*mix64(2n) + by*mix64(2n+1) mod 2^64, n = y*L+x,
// bit = (sigma+1)/2, mix64 = splitmix64 finaliser (full lattice only).
static inline uint64_t mix64(uint64_t z) {
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
uint64_t kpzo_state_hash(void* h) {
    Oracle* o = (Oracle*)h;
    uint64_t acc = 0;       // a sum mod 2^64: any order gives the same value
    #pragma omp parallel for reduction(+ : acc) schedule(static) num_threads(o->nthreads)
    for (int64_t n = 0; n < (int64_t)o->sx.size(); ++n) {
        if (o->sx[n] == 1) acc += mix64(2 * n);
        if (o->sy[n] == 1) acc += mix64(2 * n + 1);
    }
    return acc;
}

int kpzo_openmp(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 0;
#endif
}

}  // extern "C"
