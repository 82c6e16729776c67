// segments.cuh -- segment products of a resampled frame:
// minipix stamping against a target list and 16-bit float packing and the
// low-resolution map as weighted means over the minipix.  All three are streaming
// reductions over the footprint list (idx ascending, value, weight) that is already in HBM.
//
//   seg_heads_kernel     one pass over idx: a pixel is a "head" when its minipix (idx >> 2j) differs from its
//                        predecessor's; heads are numbered by a single-pass scan (per-CTA aggregate, decoupled
//                        look-back over the CTAs' status words) -> mini_start[k], mini_id[k], n_mini
//   seg_targets_kernel   every target id is looked up in mini_id (binary search, one thread per target)
//                        -> mini_keep[k] = 1.  Searching the targets into the minipix list, not the reverse,
//                        keeps the 20-step searches off the streaming kernels' critical path.
//   seg_products_kernel  one warp per minipix: sums w and w v over its pixels (fixed butterfly order), writes
//                        the binary16 bits of the stamped values, compact (element i <-> idx[i]) or scattered
//                        to the dense NSIDE-256 tile layout of argus_coadd.
#pragma once
#include <cuda_fp16.h>

#include "common.cuh"

#define SEG_ROUNDS 16
#define SEG_CHUNK (256 * SEG_ROUNDS)   // pixels per CTA of the head scan

#define SEG_FLAG_A (1ull << 62)        // status word holds the CTA's own head count
#define SEG_FLAG_P (2ull << 62)        // status word holds the inclusive prefix up to and including the CTA
#define SEG_VALUE_MASK ((1ull << 62) - 1)

struct SegLayout {
    const long long* tiles;   // ascending NSIDE-`nside_tile` ids (argus_coadd)
    long long n_tiles;
    int mini_per_tile_log2;   // 2 (log2 nside_mini - log2 nside_tile)
    int ppt_log2;             // 2 (log2 nside - log2 nside_tile)
};

__device__ __forceinline__ unsigned long long seg_ld(const unsigned long long* p) {
    return *reinterpret_cast<const volatile unsigned long long*>(p);
}
__device__ __forceinline__ void seg_st(unsigned long long* p, unsigned long long v) {
    *reinterpret_cast<volatile unsigned long long*>(p) = v;
}

// head scan.  ctl[0] = CTA ticket, ctl[1] = n_mini (both zeroed by the host before the launch); status[] zeroed.
__global__ void __launch_bounds__(256) seg_heads_kernel(const long long* __restrict__ idx, long long n, int shift,
                                                       unsigned long long* __restrict__ ctl,
                                                       unsigned long long* __restrict__ status,
                                                       long long* __restrict__ mini_start,
                                                       long long* __restrict__ mini_id, long long cap,
                                                       long long* __restrict__ n_mini_user) {
    __shared__ unsigned int s_cta;
    __shared__ int s_cnt[SEG_ROUNDS * 8];
    __shared__ long long s_base;
    __shared__ int s_total;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) s_cta = (unsigned int)atomicAdd(&ctl[0], 1ull);   // CTAs are numbered in start order: a
    __syncthreads();                                                        // predecessor is always running or done
    const unsigned int cta = s_cta;
    const long long e0 = (long long)cta * SEG_CHUNK;

    long long m[SEG_ROUNDS];
    unsigned heads = 0;
#pragma unroll
    for (int r = 0; r < SEG_ROUNDS; ++r) {
        const long long e = e0 + r * 256 + threadIdx.x;
        const bool in = e < n;
        long long cur = in ? (__ldcs(idx + e) >> shift) : -1;
        long long prev = __shfl_up_sync(0xffffffffu, cur, 1);
        if (lane == 0) prev = (in && e > 0) ? (__ldg(idx + e - 1) >> shift) : -2;
        const bool head = in && (e == 0 || cur != prev);
        const unsigned b = __ballot_sync(0xffffffffu, head);
        m[r] = cur;
        heads |= (head ? 1u : 0u) << r;
        if (lane == 0) s_cnt[r * 8 + warp] = __popc(b);
    }
    __syncthreads();
    if (warp == 0) {
        // exclusive scan of the 128 (round, warp) counts: four per lane
        int c0 = s_cnt[lane * 4], c1 = s_cnt[lane * 4 + 1], c2 = s_cnt[lane * 4 + 2], c3 = s_cnt[lane * 4 + 3];
        int sum = c0 + c1 + c2 + c3, inc = sum;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, inc, d);
            if (lane >= d) inc += t;
        }
        int ex = inc - sum;
        s_cnt[lane * 4] = ex;
        s_cnt[lane * 4 + 1] = ex + c0;
        s_cnt[lane * 4 + 2] = ex + c0 + c1;
        s_cnt[lane * 4 + 3] = ex + c0 + c1 + c2;
        const int total = __shfl_sync(0xffffffffu, inc, 31);
        if (lane == 0) seg_st(&status[cta], (cta == 0 ? SEG_FLAG_P : SEG_FLAG_A) | (unsigned long long)total);
        // decoupled look-back, 32 predecessors per step
        long long excl = 0;
        if (cta > 0) {
            long long j = (long long)cta - 1;
            for (;;) {
                const long long q = j - lane;
                unsigned long long w = (q >= 0) ? seg_ld(&status[q]) : SEG_FLAG_P;
                while (__any_sync(0xffffffffu, (w >> 62) == 0)) w = (q >= 0) ? seg_ld(&status[q]) : SEG_FLAG_P;
                const unsigned pm = __ballot_sync(0xffffffffu, (w >> 62) == 2);
                const int first = pm ? (__ffs(pm) - 1) : 32;
                long long val = (lane <= first) ? (long long)(w & SEG_VALUE_MASK) : 0;
#pragma unroll
                for (int d = 16; d > 0; d >>= 1) val += __shfl_xor_sync(0xffffffffu, val, d);
                excl += val;
                if (pm) break;
                j -= 32;
            }
            if (lane == 0) seg_st(&status[cta], SEG_FLAG_P | (unsigned long long)(excl + total));
        }
        if (lane == 0) { s_base = excl; s_total = total; }
    }
    __syncthreads();
    const long long base = s_base;
#pragma unroll
    for (int r = 0; r < SEG_ROUNDS; ++r) {
        const bool head = (heads >> r) & 1u;
        const unsigned b = __ballot_sync(0xffffffffu, head);
        if (head) {
            const long long k = base + s_cnt[r * 8 + warp] + __popc(b & ((1u << lane) - 1u));
            if (k <= cap && mini_start) mini_start[k] = e0 + r * 256 + threadIdx.x;
            if (k < cap && mini_id) mini_id[k] = m[r];
        }
    }
    if (threadIdx.x == 0 && cta == gridDim.x - 1) {
        const long long nm = base + s_total;
        ctl[1] = (unsigned long long)nm;
        if (n_mini_user) *n_mini_user = nm;
        if (nm <= cap && mini_start) mini_start[nm] = n;   // sentinel: end of the last minipix
    }
}

__global__ void __launch_bounds__(256) seg_targets_kernel(const long long* __restrict__ targets, long long n_targets,
                                                         const long long* __restrict__ mini_id,
                                                         const unsigned long long* __restrict__ ctl, long long cap,
                                                         unsigned char* __restrict__ keep) {
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    if (i >= n_targets) return;
    const long long nm = min((long long)ctl[1], cap);
    const long long t = targets[i];
    long long lo = 0, hi = nm - 1;
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

template <bool DENSE>
__global__ void __launch_bounds__(256, 6) seg_products_kernel(
    const long long* __restrict__ mini_start, const long long* __restrict__ mini_id,
    const unsigned char* __restrict__ keep, const unsigned long long* __restrict__ ctl, long long cap,
    const long long* __restrict__ idx, const float* __restrict__ value, const float* __restrict__ weight, int shift,
    SegLayout lay, unsigned short* __restrict__ seg16, float* __restrict__ mini_value, float* __restrict__ mini_weight) {
    const int lane = threadIdx.x & 31;
    const long long nw = (long long)gridDim.x * 8;
    const long long nm = min((long long)ctl[1], cap);
    const int full = 1 << shift;
    for (long long k = (long long)blockIdx.x * 8 + (threadIdx.x >> 5); k < nm; k += nw) {
        const long long s = mini_start[k], e = mini_start[k + 1];
        const int cnt = (int)(e - s);
        const bool kp = keep ? (keep[k] != 0) : true;
        long long dbase = -1;
        if (DENSE) {
            const long long mid_ = mini_id[k], key = mid_ >> lay.mini_per_tile_log2;
            long long lo = 0, hi = lay.n_tiles - 1;
            while (lo <= hi) {
                const long long mid = (lo + hi) >> 1, tv = lay.tiles[mid];
                if (tv == key) {
                    dbase = (mid << lay.ppt_log2) + ((mid_ & ((1ll << lay.mini_per_tile_log2) - 1)) << shift);
                    break;
                }
                if (tv < key) lo = mid + 1; else hi = mid - 1;
            }
        }
        float sw = 0.0f, swv = 0.0f;
        for (int q = lane; q < cnt; q += 32) {
            const float v = __ldcs(value + s + q), w = __ldcs(weight + s + q);
            sw += w;
            swv = fmaf(w, v, swv);
            if (seg16) {
                const unsigned short h = kp ? seg_f2h(v) : (unsigned short)0;
                if (DENSE) {
                    if (dbase >= 0) {
                        const long long off = (cnt == full) ? (long long)q : (idx[s + q] & (long long)(full - 1));
                        seg16[dbase + off] = h;
                    }
                } else {
                    seg16[s + q] = h;
                }
            }
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            sw += __shfl_xor_sync(0xffffffffu, sw, d);
            swv += __shfl_xor_sync(0xffffffffu, swv, d);
        }
        if (lane == 0) {
            if (mini_weight) mini_weight[k] = sw;
            if (mini_value) mini_value[k] = (sw != 0.0f) ? swv / sw : 0.0f;
        }
    }
}
