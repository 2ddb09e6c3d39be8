// kpz_aux_kernels.cuh -- the kernels of libkpz_b200.so that are not the update kernel (included by kpz.cu only):
//   kpz_fill_flat_kernel       flat zig-zag start.
//   kpz_row0_prefix_kernel,    height reconstruction (eq. 3) as a per-column chunk monoid and the exact
//   kpz_column_chunk_kernel,   integer sums of h and h^2 (eq. 4).
//   kpz_combine_kernel
//   kpz_row_inc_kernel, kpz_profile_fft_kernel, kpz_spectrum_average_kernel   axis power spectrum (eq. 15-16).
//   pack / unpack / hash / validation kernels for the parity and checkpoint calls of include/kpz.h.
#pragma once
#include "kpz_device.cuh"

namespace kpz {

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
        if (x > 0u) s += (int32_t)(((planeX[x >> 5] >> (x & 31u)) & 1u) << 1) - 1;    // sigma_x(x, 0)
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
        if (x > 0u) run += (int32_t)(((planeX[x >> 5] >> (x & 31u)) & 1u) << 1) - 1;
        out[x] = run;                         // h(x,0) - h(0,0)
    }
}

// Column-chunk kernel.  grid (ceil(W/128), n_chunks, R), block 128: one THREAD owns one word-column (32 columns)
// of one chunk of rows_per_chunk <= 1024 rows (a multiple of 32).  Per 32 rows it loads 32 words (coalesced across
// the lanes of a warp), transposes the 32x32 bit block in registers so that each column becomes one word (bit k =
// row k), and walks every column 8 rows at a time through a 256-entry table in shared memory: a byte b of sigma_y
// bits (bit k set <=> step +1) has exit S0 = l_7, S1 = sum l_k, S2 = sum l_k^2 with l_k = sum_{j<=k} (+-1), and a
// leaf of n = 8 rows entered at height B contributes n*B + S1 and n*B^2 + 2*B*S1 + S2.  Row 0 of the lattice
// carries no sigma_y step (eq. 3): chunk 0 is walked as if it did and corrected per column afterwards
// (l = l' - s0:  sum l = sum l' - n*s0,  sum l^2 = sum l'^2 - 2*s0*sum l' + n).
// All chunk-relative sums fit 32 bits: |l| <= 1024, sum l^2 <= 2^30.
__device__ __forceinline__ void transpose32x32(uint32_t (&a)[32]) {
    // after the call: bit k of a[c] = bit c of the former a[k]
#pragma unroll
    for (int j = 16, it = 0; it < 5; ++it, j >>= 1) {
        const uint32_t m = (j == 16) ? 0x0000FFFFu : (j == 8) ? 0x00FF00FFu : (j == 4) ? 0x0F0F0F0Fu
                         : (j == 2) ? 0x33333333u : 0x55555555u;
#pragma unroll
        for (int k = 0; k < 32; ++k) {
            if ((k & j) == 0) {
                const uint32_t t = ((a[k] >> j) ^ a[k + j]) & m;
                a[k] ^= t << j;
                a[k + j] ^= t;
            }
        }
    }
}

__global__ void __launch_bounds__(128) kpz_column_chunk_kernel(const uint32_t* __restrict__ lattice,
                                                               uint64_t plane_words, uint32_t L, uint32_t W,
                                                               uint32_t rows_per_chunk, int32_t* __restrict__ cS0,
                                                               int32_t* __restrict__ cS1, int32_t* __restrict__ cS2,
                                                               uint32_t n_rows, uint32_t row0_is_lattice_row0) {
    // n_rows stored rows are walked (L for a whole lattice, the owned rows of a slab); L is the number of columns.
    // row0_is_lattice_row0 = 0 for a slab that does not start at lattice row 0: its first row is an ordinary step.
    // One 256-entry copy for the whole CTA.  (A copy per bank, lut[32 * byte + lane], removes the 1.6e8 bank
    // conflicts of a measurement at L = 2^17 but costs an index shift and 32 KB per CTA: 1.76 ms against 1.54 ms,
    // the kernel is bound by the ALU pipe at 70 %, not by the table -- measured in round 2 and dropped.)
    __shared__ uint32_t lut[256];      // (S0 & 0xFF) | (S1 & 0xFF) << 8 | S2 << 16
    for (uint32_t b = threadIdx.x; b < 256u; b += blockDim.x) {
        int l = 0, s1 = 0, s2 = 0;
        for (int k = 0; k < 8; ++k) {
            l += ((b >> k) & 1u) ? 1 : -1;
            s1 += l;
            s2 += l * l;
        }
        lut[b] = ((uint32_t)l & 0xFFu) | (((uint32_t)s1 & 0xFFu) << 8) | ((uint32_t)s2 << 16);
    }
    __syncthreads();
    const uint32_t wcol = blockIdx.x * 128u + threadIdx.x;
    if (wcol >= W) return;
    const uint32_t chunk = blockIdx.y, replica = blockIdx.z, n_chunks = gridDim.y;
    const uint32_t* planeY = lattice + (size_t)replica * 2u * plane_words + plane_words;
    const uint32_t y_begin = chunk * rows_per_chunk;
    const uint32_t y_end = min(n_rows, y_begin + rows_per_chunk);
    int32_t B[32], s1[32], s2[32];
#pragma unroll
    for (int c = 0; c < 32; ++c) { B[c] = 0; s1[c] = 0; s2[c] = 0; }
    uint32_t first_row = 0u;
#pragma unroll 1
    for (uint32_t yb = y_begin; yb < y_end; yb += 32u) {
        uint32_t a[32];
#pragma unroll
        for (int k = 0; k < 32; ++k) a[k] = __ldg(planeY + (size_t)(yb + (uint32_t)k) * W + wcol);
        if (yb == 0u) first_row = a[0];
        transpose32x32(a);
#pragma unroll
        for (int c = 0; c < 32; ++c) {
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const uint32_t e = lut[(a[c] >> (8 * q)) & 0xFFu];
                const int32_t S0 = (int32_t)(int8_t)(e & 0xFFu), S1 = (int32_t)(int8_t)((e >> 8) & 0xFFu);
                const int32_t S2 = (int32_t)(e >> 16);
                const int32_t t = 8 * B[c] + S1;
                s1[c] += t;
                s2[c] += B[c] * (t + S1) + S2;
                B[c] += S0;
            }
        }
    }
    const int32_t n = (int32_t)(y_end - y_begin);
    const size_t o = ((size_t)replica * n_chunks + chunk) * L + (size_t)wcol * 32u;
#pragma unroll
    for (int c = 0; c < 32; ++c) {
        if (chunk == 0u && row0_is_lattice_row0) {
            const int32_t s0 = ((first_row >> c) & 1u) ? 1 : -1;
            s2[c] += -2 * s0 * s1[c] + n;
            s1[c] -= n * s0;
            B[c] -= s0;
        }
        cS0[o + c] = B[c];
        cS1[o + c] = s1[c];
        cS2[o + c] = s2[c];
    }
}

// grid (ceil(L/256), R), block 256: one thread per column; out[replica][4] += {lo(S1), hi(S1), lo(S2), hi(S2)}
__global__ void __launch_bounds__(256) kpz_combine_kernel(const int32_t* __restrict__ base,
                                                          const int32_t* __restrict__ cS0,
                                                          const int32_t* __restrict__ cS1,
                                                          const int32_t* __restrict__ cS2, uint32_t L,
                                                          uint32_t n_chunks, uint32_t rows_per_chunk,
                                                          unsigned long long* __restrict__ msum,
                                                          long long* __restrict__ colsum, uint32_t colsum_replica,
                                                          uint32_t n_rows) {
    const uint32_t replica = blockIdx.y;
    const uint32_t x = blockIdx.x * 256u + threadIdx.x;
    long long a1 = 0, a2 = 0;
    if (x < L) {
        long long B = base[(size_t)replica * L + x];
        for (uint32_t c = 0; c < n_chunks; ++c) {
            const uint32_t y_begin = c * rows_per_chunk;
            if (y_begin >= n_rows) break;
            const long long n = (long long)(min(n_rows, y_begin + rows_per_chunk) - y_begin);
            const size_t o = ((size_t)replica * n_chunks + c) * L + x;
            const long long S1 = cS1[o], S2 = cS2[o];
            a1 += n * B + S1;
            a2 += n * B * B + 2 * B * S1 + S2;
            B += cS0[o];
        }
        if (colsum != nullptr && replica == colsum_replica) colsum[x] = a1;   // sum_y (h(x,y) - h00)
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
// Power spectrum along the two lattice axes (eq. 15-16).  With
// h(k) = (1/L) sum_x [h(x) - <h>] exp(i k.x), the modes on the k_x axis depend on the surface only through its
// column sums c(x) = sum_y h(x,y) and those on the k_y axis only through its row sums r(y) = sum_x h(x,y):
// h(k_x, 0) = (1/L) sum_x c(x) exp(i k_x x).  The column sums come out of kpz_combine_kernel; the row sums are
// r(0) = sum_x base(x) and r(y) = r(y-1) + 2*popc(row y of sigma_y) - L.  Both profiles are exact integers.
// ------------------------------------------------------------------------------------------------------------
// one warp per row: inc[y] = sum_x sigma_y(x,y) = 2*popc - L
__global__ void __launch_bounds__(256) kpz_row_inc_kernel(const uint32_t* __restrict__ lattice, uint64_t plane_words,
                                                          uint32_t replica, uint32_t L, uint32_t W,
                                                          int32_t* __restrict__ inc) {
    const uint32_t* planeY = lattice + (size_t)replica * 2u * plane_words + plane_words;
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t warps = (gridDim.x * blockDim.x) >> 5;
    for (uint32_t y = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; y < L; y += warps) {
        uint32_t c = 0;
        for (uint32_t k = lane; k < W; k += 32u) c += __popc(__ldg(planeY + (size_t)y * W + k));
#pragma unroll
        for (int sft = 16; sft > 0; sft >>= 1) c += __shfl_xor_sync(0xFFFFFFFFu, c, sft);
        if (lane == 0u) inc[y] = (int32_t)(2u * c) - (int32_t)L;
    }
}

__device__ __forceinline__ long long block_sum_ll(long long v, long long* red) {
    // sum over the 1024 threads of the block, returned to every thread
#pragma unroll
    for (int sft = 16; sft > 0; sft >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, sft);
    __syncthreads();
    if ((threadIdx.x & 31u) == 0u) red[threadIdx.x >> 5] = v;
    __syncthreads();
    long long t = 0;
    for (int w = 0; w < 32; ++w) t += red[w];
    return t;
}

// grid 2 (block 0: column profile / k_x axis, block 1: row profile / k_y axis), block 1024.  Builds the profile
// relative to h00, removes an integer approximation of its mean (a constant only changes the k = 0 mode, which
// is 0 by definition; removing it keeps the rounding of the transform small), runs an in-place radix-2
// decimation-in-time FFT in fp64 on `buf` (twiddles from sincospi), and writes S(k) = |X(k)|^2 / L^2 for
// k = 0 .. L/2.  L must be a power of two.
__global__ void __launch_bounds__(1024) kpz_profile_fft_kernel(const long long* __restrict__ colsum,
                                                               const int32_t* __restrict__ base,
                                                               const int32_t* __restrict__ inc,
                                                               long long* __restrict__ prof, double2* __restrict__ buf,
                                                               double* __restrict__ Sdir, uint32_t L, uint32_t logL) {
    __shared__ long long red[32];
    __shared__ long long seg[1024];
    const uint32_t dir = blockIdx.x, tid = threadIdx.x;
    long long* p = prof + (size_t)dir * L;
    double2* b = buf + (size_t)dir * L;
    const uint32_t per = (L + 1023u) / 1024u;
    const uint32_t i0 = tid * per, i1 = min(L, i0 + per);
    if (dir == 0u) {
        for (uint32_t i = tid; i < L; i += 1024u) p[i] = colsum[i];
    } else {
        // r(0) = sum_x base(x); r(y) = r(y-1) + inc(y): block scan over contiguous segments
        long long sb = 0;
        for (uint32_t i = tid; i < L; i += 1024u) sb += base[i];
        const long long r0 = block_sum_ll(sb, red);
        long long s = 0;
        for (uint32_t i = i0; i < i1; ++i) s += (i == 0u) ? 0 : inc[i];
        seg[tid] = s;
        __syncthreads();
        for (uint32_t d = 1; d < 1024u; d <<= 1) {
            const long long v = (tid >= d) ? seg[tid - d] : 0;
            __syncthreads();
            seg[tid] += v;
            __syncthreads();
        }
        long long run = r0 + seg[tid] - s;
        for (uint32_t i = i0; i < i1; ++i) {
            run += (i == 0u) ? 0 : inc[i];
            p[i] = run;
        }
    }
    __syncthreads();
    if (logL == 0u) return;          // profiles only
    long long sl = 0;
    for (uint32_t i = tid; i < L; i += 1024u) sl += p[i];
    const long long mean = block_sum_ll(sl, red) / (long long)L;
    for (uint32_t i = tid; i < L; i += 1024u) {
        const uint32_t j = __brev(i) >> (32u - logL);
        b[j] = make_double2((double)(p[i] - mean), 0.0);
    }
    __syncthreads();
    for (uint32_t s = 1; s <= logL; ++s) {
        const uint32_t half = 1u << (s - 1u);
        for (uint32_t t = tid; t < (L >> 1); t += 1024u) {
            const uint32_t j = t & (half - 1u);
            const uint32_t lo = ((t >> (s - 1u)) << s) + j, hi = lo + half;
            double sn, cs;
            sincospi(-(double)j / (double)half, &sn, &cs);
            const double2 u = b[lo], v = b[hi];
            const double2 w = make_double2(v.x * cs - v.y * sn, v.x * sn + v.y * cs);
            b[lo] = make_double2(u.x + w.x, u.y + w.y);
            b[hi] = make_double2(u.x - w.x, u.y - w.y);
        }
        __syncthreads();
    }
    const double inv = 1.0 / ((double)L * (double)L);
    for (uint32_t k = tid; k <= (L >> 1); k += 1024u)
        Sdir[(size_t)dir * ((L >> 1) + 1u) + k] = (k == 0u) ? 0.0 : (b[k].x * b[k].x + b[k].y * b[k].y) * inv;
}

// "averaging over x and y directions": S(k) = (S(k,0) + S(0,k)) / 2
__global__ void kpz_spectrum_average_kernel(const double* __restrict__ Sdir, double* __restrict__ S, uint32_t n) {
    const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) S[k] = 0.5 * (Sdir[k] + Sdir[n + k]);
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
        const uint32_t bxv = (planeX[(size_t)y * W + (x >> 5)] >> (x & 31u)) & 1u;
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
            // both planes: line = y, c = x
            if (sx[(size_t)line * L + c] > 0) wx |= 1u << b;
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
        const uint32_t wx = planeX[t];      // same row, same columns
        for (uint32_t b = 0; b < 32u; ++b) {
            const uint32_t c = 32u * k + b;
            if ((wy >> b) & 1u) acc += mix64(2ull * ((uint64_t)line * L + c) + 1ull);
            if ((wx >> b) & 1u) acc += mix64(2ull * ((uint64_t)line * L + c));
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

// ------------------------------------------------------------------------------------------------------------
// Slab helpers: per-column step total of a slab's owned rows, and the entry height of a slab
// from the row-0 prefix and the totals of the slabs below it.
// ------------------------------------------------------------------------------------------------------------
__global__ void kpz_slab_totals_kernel(const int32_t* __restrict__ cS0, uint32_t L, uint32_t n_chunks, uint32_t rows_per_chunk,
                                       uint32_t n_rows, int32_t* __restrict__ tot) {
    const uint32_t x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= L) return;
    int32_t t = 0;
    for (uint32_t c = 0; c < n_chunks && c * rows_per_chunk < n_rows; ++c) t += cS0[(size_t)c * L + x];
    tot[x] = t;
}

// base[x] = base0[x] + sum_{r' < slab} tot_all[r'][x]
__global__ void kpz_slab_base_kernel(const int32_t* __restrict__ base0, const int32_t* __restrict__ tot_all, uint32_t L,
                                     uint32_t slab, int32_t* __restrict__ base) {
    const uint32_t x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= L) return;
    int32_t b = base0[x];
    for (uint32_t r = 0; r < slab; ++r) b += tot_all[(size_t)r * L + x];
    base[x] = b;
}

}  // namespace kpz
