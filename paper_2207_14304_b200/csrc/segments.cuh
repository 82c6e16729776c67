// segments.cuh -- segment products of a resampled frame:
// minipix stamping against a target list and 16-bit float packing and the
// low-resolution map as weighted means over the minipix.  All three are streaming
// reductions over the footprint list (idx ascending, value, weight) that is already in HBM.
//
//   seg_flags_kernel     one pass over idx: a pixel is a "head" when its minipix (idx >> 2j) differs from its
//   seg_scan_kernel      predecessor's; one flag bit per pixel + head count per 4096-pixel chunk, scan of the
//   seg_heads_kernel     counts, then mini_start[k] (position of the k-th head), mini_id[k], n_mini
//   seg_targets_kernel   every target id is looked up in mini_id (binary search, one thread per target)
//                        -> mini_keep[k] = 1.  Searching the targets into the minipix list, not the reverse,
//                        keeps the 20-step searches off the streaming kernels' critical path.
//   seg_products_kernel  one warp per four minipix: sums w and w v over their pixels (fixed butterfly order), writes
//                        the binary16 bits of the stamped values, compact (element i <-> idx[i]) or scattered
//                        to the dense NSIDE-256 tile layout of argus_coadd.
#pragma once
#include <cuda_fp16.h>

#include "common.cuh"

#define SEG_ROUNDS 8
#define SEG_CHUNK (256 * SEG_ROUNDS)   // pixels per CTA of the head scan

struct SegLayout {
    const long long* tiles;   // ascending NSIDE-`nside_tile` ids (argus_coadd)
    long long n_tiles;
    int mini_per_tile_log2;   // 2 (log2 nside_mini - log2 nside_tile)
    int ppt_log2;             // 2 (log2 nside - log2 nside_tile)
};

// Heads, pass 1: one streaming pass over idx.  Pixel e is a head when its minipix differs from pixel e-1's.  Writes
// one flag bit per pixel (bits[e / 32], 1/64 of the bytes read) and the number of heads of every 4096-pixel chunk.
// (A single-pass scan with decoupled look-back was measured first: its CTAs spent 45 % of their life polling their
// predecessors' status words, 0.28 ms for 359 MB; the three free-running kernels below take a quarter of that.)
__global__ void __launch_bounds__(256) seg_flags_kernel(const long long* __restrict__ idx, long long n, int shift,
                                                       unsigned int* __restrict__ bits,
                                                       unsigned int* __restrict__ counts) {
    __shared__ long long s_last[SEG_ROUNDS * 8];
    __shared__ int s_cnt[8];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long e0 = (long long)blockIdx.x * SEG_CHUNK;
    long long m[SEG_ROUNDS];
    long long before = -2;
    if (threadIdx.x == 0 && e0 > 0) before = __ldg(idx + e0 - 1) >> shift;
#pragma unroll
    for (int r = 0; r < SEG_ROUNDS; ++r) {   // all loads first: 16 in flight per thread
        const long long e = e0 + r * 256 + threadIdx.x;
        m[r] = (e < n) ? (__ldcs(idx + e) >> shift) : -1;
    }
    if (lane == 31) {
#pragma unroll
        for (int r = 0; r < SEG_ROUNDS; ++r) s_last[r * 8 + warp] = m[r];
    }
    __syncthreads();
    int cnt = 0;
#pragma unroll
    for (int r = 0; r < SEG_ROUNDS; ++r) {
        const long long e = e0 + r * 256 + threadIdx.x;
        long long prev = __shfl_up_sync(0xffffffffu, m[r], 1);
        if (lane == 0) prev = (r * 8 + warp > 0) ? s_last[r * 8 + warp - 1] : before;
        const bool head = e < n && (e == 0 || m[r] != prev);
        const unsigned b = __ballot_sync(0xffffffffu, head);
        if (lane == 0) bits[(long long)blockIdx.x * (SEG_CHUNK / 32) + r * 8 + warp] = b;
        cnt += __popc(b);
    }
    if (lane == 0) s_cnt[warp] = cnt;
    __syncthreads();
    if (threadIdx.x == 0) {
        int t = 0;
#pragma unroll
        for (int i = 0; i < 8; ++i) t += s_cnt[i];
        counts[blockIdx.x] = (unsigned int)t;
    }
    // the scan reads counts in groups of 32 chunks: the last CTA zeroes the rest of the last group
    if (blockIdx.x == gridDim.x - 1 && warp == 1 && gridDim.x + lane < ((gridDim.x + 31u) & ~31u)) counts[gridDim.x + lane] = 0;
}

// Heads, pass 2: exclusive scan of the chunk counts at the granularity of 32 chunks (one CTA: thread t sums chunks
// 32 t .. 32 t + 31 with eight independent 16-byte loads, so a 45 M pixel frame is one round of one load latency);
// pass 3 adds the up to 31 counts in front of its own chunk.  ctl[1] = n_mini; mini_start[n_mini] = n is the
// sentinel that ends the last minipix.  `counts` is padded to a multiple of 32 chunks (zeros past n_chunks).
__global__ void __launch_bounds__(1024) seg_scan_kernel(const unsigned int* __restrict__ counts, long long n_chunks,
                                                       long long* __restrict__ offsets32,
                                                       unsigned long long* __restrict__ ctl,
                                                       long long* __restrict__ n_mini_user,
                                                       long long* __restrict__ mini_start, long long cap, long long n) {
    __shared__ long long s_w[32];
    __shared__ long long s_carry;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long n32 = (n_chunks + 31) / 32;
    long long carry = 0;
    for (long long base = 0; base < n32; base += 1024) {
        const long long g = base + threadIdx.x;
        long long v = 0;
        if (g < n32) {
            const uint4* q = reinterpret_cast<const uint4*>(counts + g * 32);
            uint4 r[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) r[i] = q[i];
#pragma unroll
            for (int i = 0; i < 8; ++i) v += (long long)r[i].x + r[i].y + r[i].z + r[i].w;
        }
        long long inc = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const long long t = __shfl_up_sync(0xffffffffu, inc, d);
            if (lane >= d) inc += t;
        }
        if (lane == 31) s_w[warp] = inc;
        __syncthreads();
        if (warp == 0) {
            long long w = s_w[lane], wi = w;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const long long t = __shfl_up_sync(0xffffffffu, wi, d);
                if (lane >= d) wi += t;
            }
            s_w[lane] = wi - w;
            if (lane == 31) s_carry = wi;
        }
        __syncthreads();
        if (g < n32) offsets32[g] = carry + s_w[warp] + inc - v;
        carry += s_carry;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const long long nm = carry;
        ctl[1] = (unsigned long long)nm;
        if (n_mini_user) *n_mini_user = nm;
        if (nm <= cap && mini_start) mini_start[nm] = n;
    }
}

// Heads, pass 3: flag bits + chunk offsets -> mini_start[k] (position of the k-th head), mini_id[k].
#define SEG_HEADS_CPB 4   // chunks per CTA of pass 3 (64 flag words each: two warps per chunk)
__global__ void __launch_bounds__(SEG_HEADS_CPB * SEG_CHUNK / 32) seg_heads_kernel(
    const unsigned int* __restrict__ bits, const unsigned int* __restrict__ counts, long long n_chunks,
    const long long* __restrict__ offsets32, const long long* __restrict__ idx, int shift,
    long long* __restrict__ mini_start, long long* __restrict__ mini_id, unsigned char* __restrict__ keep, long long cap) {
    constexpr int WPC = SEG_CHUNK / 1024;   // warps per chunk
    __shared__ int s_w[SEG_HEADS_CPB * WPC];
    __shared__ int s_front[SEG_HEADS_CPB];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const long long chunk = (long long)blockIdx.x * SEG_HEADS_CPB + warp / WPC;
    if (chunk >= n_chunks) { __syncthreads(); return; }   // whole warps leave together; the barrier count stays right
    if (warp % WPC == 0) {   // heads of the chunks in front of this one inside its group of 32
        int f = (lane < (int)(chunk & 31)) ? (int)counts[(chunk & ~31ll) + lane] : 0;
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) f += __shfl_xor_sync(0xffffffffu, f, d);
        if (lane == 0) s_front[warp / WPC] = f;
    }
    unsigned word = bits[chunk * (SEG_CHUNK / 32) + (threadIdx.x & (SEG_CHUNK / 32 - 1))];
    const int c = __popc(word);
    int inc = c;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += t;
    }
    if (lane == 31) s_w[warp] = inc;
    __syncthreads();
    int wbase = 0;
#pragma unroll
    for (int i = 0; i < WPC; ++i) wbase += (i < warp % WPC) ? s_w[warp / WPC * WPC + i] : 0;
    long long k = offsets32[chunk >> 5] + s_front[warp / WPC] + wbase + inc - c;
    const long long e0 = chunk * SEG_CHUNK + (threadIdx.x & (SEG_CHUNK / 32 - 1)) * 32;
    while (word) {
        const int b = __ffs(word) - 1;
        word &= word - 1;
        const long long e = e0 + b;
        if (k <= cap && mini_start) mini_start[k] = e;
        if (k < cap && mini_id) mini_id[k] = __ldg(idx + e) >> shift;
        if (k < cap && keep) keep[k] = 0;   // seg_targets_kernel sets the kept ones afterwards
        ++k;
    }
}

__global__ void __launch_bounds__(256) seg_targets_kernel(const long long* __restrict__ targets, long long n_targets,
                                                         const long long* __restrict__ mini_id,
                                                         const unsigned long long* __restrict__ ctl, long long cap,
                                                         unsigned char* __restrict__ keep) {
    // 256 evenly spaced entries of mini_id in shared memory take the first 8 of the ~20 search steps off the
    // dependent chain of L2 reads (the kernel is that chain: 13 us -> 9 us for 14 k targets in 703 k minipix)
    __shared__ long long s_tab[256];
    const long long nm = min((long long)ctl[1], cap);
    if (nm <= 0) return;
    s_tab[threadIdx.x] = mini_id[(long long)(threadIdx.x + 1) * nm / 257];
    __syncthreads();
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    if (i >= n_targets) return;
    const long long t = targets[i];
    int a = 0, b = 256;                    // first table entry >= t
    while (a < b) {
        const int mid = (a + b) >> 1;
        if (s_tab[mid] < t) a = mid + 1; else b = mid;
    }
    long long lo = (a == 0) ? 0 : (long long)a * nm / 257;            // position of table entry a - 1
    long long hi = (a == 256) ? nm - 1 : (long long)(a + 1) * nm / 257;   // position of table entry a
    while (lo <= hi) {
        const long long mid = (lo + hi) >> 1, v = mini_id[mid];
        if (v == t) { keep[mid] = 1; return; }
        if (v < t) lo = mid + 1; else hi = mid - 1;
    }
}

// float -> binary16 bits, round to nearest even; finite values clamped to +-65504, NaN -> 0x7e00 (DESIGN.md R-S2)
__device__ __forceinline__ unsigned short seg_f2h(float v) {
    const float c = fminf(fmaxf(v, -65504.0f), 65504.0f);
    const unsigned short h = __half_as_ushort(__float2half_rn(c));
    return (v != v) ? (unsigned short)0x7e00 : h;
}

// row-major position iy * side + ix of an in-tile nested index (ix = even bits, iy = odd bits)
__device__ __forceinline__ long long seg_raster(long long local, int side_log2) {
    return (long long)compact_even_bits((unsigned long long)local) +
           ((long long)compact_even_bits((unsigned long long)local >> 1) << side_log2);
}

// dense-layout base slot of minipix `mid_` (or -1 when its tile is absent)
__device__ __forceinline__ long long seg_dense_base(const SegLayout& lay, long long mid_, int shift, bool raster) {
    const long long key = mid_ >> lay.mini_per_tile_log2;
    long long lo = 0, hi = lay.n_tiles - 1;
    while (lo <= hi) {
        const long long mid = (lo + hi) >> 1, tv = lay.tiles[mid];
        if (tv == key) {
            const long long local = (mid_ & ((1ll << lay.mini_per_tile_log2) - 1)) << shift;   // minipix' first pixel
            return (mid << lay.ppt_log2) + (raster ? seg_raster(local, lay.ppt_log2 >> 1) : local);
        }
        if (tv < key) lo = mid + 1; else hi = mid - 1;
    }
    return -1;
}

#define SEG_GROUP 4   // minipix per warp iteration: their pixels are adjacent in the list, 4 x 4 loads in flight per lane

// Sum of eight per-lane values over the warp in 10 shuffles: each butterfly step halves the number of values a lane
// carries (lane bit 4 picks a[0..3] / a[4..7], bit 3 the pair, bit 2 the value), the last two steps are plain.
// Returns, in every lane, the total of value q = 4 (lane >> 4 & 1) + 2 (lane >> 3 & 1) + (lane >> 2 & 1).  Fixed order.
__device__ __forceinline__ float seg_reduce8(const float (&a)[8], int lane) {
    float b[4], c[2];
    const bool u4 = lane & 16, u3 = lane & 8, u2 = lane & 4;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float send = u4 ? a[k] : a[k + 4], keep = u4 ? a[k + 4] : a[k];
        b[k] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
    }
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        const float send = u3 ? b[k] : b[k + 2], keep = u3 ? b[k + 2] : b[k];
        c[k] = keep + __shfl_xor_sync(0xffffffffu, send, 8);
    }
    float d = (u2 ? c[1] : c[0]) + __shfl_xor_sync(0xffffffffu, u2 ? c[0] : c[1], 4);
    d += __shfl_xor_sync(0xffffffffu, d, 2);
    d += __shfl_xor_sync(0xffffffffu, d, 1);
    return d;
}

// DENSE: 0 = seg16 element i <-> idx[i]; 1 = tile-dense layout, nested order inside a tile; 2 = tile-dense, row-major
template <int DENSE>
__global__ void __launch_bounds__(256, 4) seg_products_kernel(
    const long long* __restrict__ mini_start, const long long* __restrict__ mini_id,
    const unsigned char* __restrict__ keep, const unsigned long long* __restrict__ ctl, long long cap,
    const long long* __restrict__ idx, const float* __restrict__ value, const float* __restrict__ weight, int shift,
    SegLayout lay, unsigned short* __restrict__ seg16, float* __restrict__ mini_value, float* __restrict__ mini_weight) {
    const int lane = threadIdx.x & 31;
    const long long nw = (long long)gridDim.x * 8;
    const long long nm = min((long long)ctl[1], cap);
    const long long full = 1ll << shift;   // pixels per minipix: up to 4^29 (nside 2^29, nside_mini 1)
    for (long long kb = ((long long)blockIdx.x * 8 + (threadIdx.x >> 5)) * SEG_GROUP; kb < nm; kb += nw * SEG_GROUP) {
        // lanes 0..4: starts of the group's minipix (mini_start[nm] is the sentinel); lanes 0..3: keep flag, dense base
        const long long st = (lane <= SEG_GROUP) ? mini_start[min(kb + lane, nm)] : 0;
        int kp_l = 1;
        long long db_l = -1;
        if (lane < SEG_GROUP && kb + lane < nm) {
            if (keep) kp_l = keep[kb + lane] != 0;
            if (DENSE) db_l = seg_dense_base(lay, mini_id[kb + lane], shift, DENSE == 2);
        }
        const long long s0 = __shfl_sync(0xffffffffu, st, 0);
        const int rel_l = (int)min(st - s0, (long long)0x3fffffff);   // pixels of the group lie in [s0, s0 + rel[4])
        int rel[SEG_GROUP + 1];
#pragma unroll
        for (int i = 0; i <= SEG_GROUP; ++i) rel[i] = __shfl_sync(0xffffffffu, rel_l, i);
        const unsigned kpm = __ballot_sync(0xffffffffu, kp_l != 0);
        bool small = true;
#pragma unroll
        for (int i = 0; i < SEG_GROUP; ++i) small = small && (rel[i + 1] - rel[i] <= 64);
        small = small && (__shfl_sync(0xffffffffu, st, SEG_GROUP) - s0 <= 64 * SEG_GROUP);   // rel is clamped: be exact
        const float* vb = value + s0;
        const float* wb = weight + s0;
        float acc[8];
        if (small) {
            // every minipix of the group has at most 64 pixels (the paper's case, 4^3): all loads issued up front,
            // 32-bit offsets from the group's first pixel
            float v[SEG_GROUP][2], w[SEG_GROUP][2];
            int left[SEG_GROUP];                           // pixels of minipix i from this lane's first one on
#pragma unroll
            for (int i = 0; i < SEG_GROUP; ++i) {
                const float* vi = vb + (rel[i] + lane);    // one 64-bit address per minipix and array; the second
                const float* wi = wb + (rel[i] + lane);    // pixel of the lane is 128 B further
                left[i] = rel[i + 1] - rel[i] - lane;
                v[i][0] = (left[i] > 0) ? __ldcs(vi) : 0.0f;
                w[i][0] = (left[i] > 0) ? __ldcs(wi) : 0.0f;
                v[i][1] = (left[i] > 32) ? __ldcs(vi + 32) : 0.0f;
                w[i][1] = (left[i] > 32) ? __ldcs(wi + 32) : 0.0f;
            }
#pragma unroll
            for (int i = 0; i < SEG_GROUP; ++i) {
                acc[2 * i] = w[i][0] + w[i][1];
                acc[2 * i + 1] = fmaf(w[i][1], v[i][1], w[i][0] * v[i][0]);
                if (seg16) {
                    const bool kp = (kpm >> i) & 1u;
                    const unsigned short h0 = kp ? seg_f2h(v[i][0]) : (unsigned short)0;
                    const unsigned short h1 = kp ? seg_f2h(v[i][1]) : (unsigned short)0;
                    if (DENSE) {
                        const long long dbase = __shfl_sync(0xffffffffu, db_l, i);
                        if (dbase >= 0) {
                            const bool complete = rel[i + 1] - rel[i] == full;
                            const long long* ii = idx + s0 + (rel[i] + lane);
                            long long o0 = complete ? (long long)lane : (left[i] > 0 ? (ii[0] & (full - 1)) : 0);
                            long long o1 = complete ? (long long)(lane + 32) : (left[i] > 32 ? (ii[32] & (full - 1)) : 0);
                            if (DENSE == 2) { o0 = seg_raster(o0, lay.ppt_log2 >> 1); o1 = seg_raster(o1, lay.ppt_log2 >> 1); }
                            if (left[i] > 0) seg16[dbase + o0] = h0;
                            if (left[i] > 32) seg16[dbase + o1] = h1;
                        }
                    } else {
                        unsigned short* oi = seg16 + s0 + (rel[i] + lane);
                        if (left[i] > 0) oi[0] = h0;
                        if (left[i] > 32) oi[32] = h1;
                    }
                }
            }
        } else {
#pragma unroll
            for (int i = 0; i < SEG_GROUP; ++i) {
                const long long si = __shfl_sync(0xffffffffu, st, i);
                const long long cnt = __shfl_sync(0xffffffffu, st, i + 1) - si;
                const bool kp = (kpm >> i) & 1u;
                const long long dbase = DENSE ? __shfl_sync(0xffffffffu, db_l, i) : 0;
                float sw = 0.0f, swv = 0.0f;
                for (long long q = lane; q < cnt; q += 32) {
                    const float vv = __ldcs(value + si + q), ww = __ldcs(weight + si + q);
                    sw += ww;
                    swv = fmaf(ww, vv, swv);
                    if (seg16) {
                        const unsigned short hb = kp ? seg_f2h(vv) : (unsigned short)0;
                        if (DENSE) {
                            if (dbase >= 0) {
                                long long o = (cnt == full) ? q : (idx[si + q] & (full - 1));
                                if (DENSE == 2) o = seg_raster(o, lay.ppt_log2 >> 1);
                                seg16[dbase + o] = hb;
                            }
                        } else {
                            seg16[si + q] = hb;
                        }
                    }
                }
                acc[2 * i] = sw;
                acc[2 * i + 1] = swv;
            }
        }
        const float tot = seg_reduce8(acc, lane);                       // lanes with bit 2 clear: sum w; set: sum w v
        const float oth = __shfl_xor_sync(0xffffffffu, tot, 4);
        const int i = ((lane >> 4) & 1) * 2 + ((lane >> 3) & 1);
        if ((lane & 7) == 0 && kb + i < nm) {
            if (mini_weight) mini_weight[kb + i] = tot;
            if (mini_value) mini_value[kb + i] = (tot != 0.0f) ? oth / tot : 0.0f;
        }
    }
}
