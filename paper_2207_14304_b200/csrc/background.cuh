// background.cuh -- median-filtered background / noise map and source detection on the calibrated frame
// (DESIGN.md section 11): the two GPU stages the paper runs between calibration and
// resampling (PAPER.md:193-194 Table 2, :135; "intermediate background and noise maps" :109).  Calibration is
// fused into both passes when the frame arrives as raw + masters (the calibrated frame never exists in HBM).
//
//   bg_cells_kernel    one CTA per B x B cell (B <= 64): the cell's pixels live in registers (16 per thread) as
//                      order-preserving 32-bit keys; the two central order statistics are found EXACTLY by a
//                      multi-level counting select (256-bin shared histogram over the live key range, CTA-wide
//                      scan, descend into the bin that holds the rank: 8 bits per level), started at the common
//                      prefix of the cell's min and max and finished by ranking the survivors once 32 or fewer
//                      remain.  Same again on |v - med| for the MAD noise estimate.
//   bg_filter_kernel   3x3 median over the valid cells of the grid (one thread per cell).
//   det_tiles_kernel   one CTA per 64 x 32-pixel tile: s = cal - bkg(x, y) for the tile + 1-pixel apron in shared
//                      memory, thresholded raster-first local maxima, 3x3 flux and centroid; records go to a
//                      scratch list at an atomically reserved base, (base, count) per tile.
//   det_order_kernel   one CTA per tile row: start of the row in the catalogue from the per-row counts, then ranks the row's
//                      records by raster index and writes them to their final position (catalogue order = ascending
//                      y * W + x, R-D6).
//   det_scan_kernel    exclusive scan of per-block counts (argus_subtract_tiles).
#pragma once
#include "resample.cuh"

#define BG_THREADS 256
#define BG_KPT 16                    // keys per thread: 256 x 16 = 4096 = 64 x 64
#define BG_SENTINEL 0xffffffffu      // masked / outside the cell: sorts after every value
#define BG_FINISH 32                 // rank the survivors directly once this few remain
#define BG_SAMPLE_MIN 24             // valid keys among the 64 sampled below which no range is guessed
#define BG_MAD_TO_SIGMA 1.4826f

struct ArgusSourceRec {              // == argus_source (argus.h)
    int x, y;
    float peak, flux, cx, cy, bkg, nse;
};

__device__ __forceinline__ unsigned bg_key(float v) {
    const unsigned u = __float_as_uint(v);
    // negative: all bits flipped, else the sign bit set
    return (v != v) ? BG_SENTINEL : (u ^ ((unsigned)((int)u >> 31) | 0x80000000u));
}
__device__ __forceinline__ float bg_unkey(unsigned k) {
    return __uint_as_float((k & 0x80000000u) ? (k ^ 0x80000000u) : ~k);
}
// ++hist[bin] when d <= span.  Written without a branch: keys outside the range count into the spare word BG_HIST_SPARE
// (never read), which the hardware folds into one increment per warp (ATOMS.POPC.INC); the compiler's form of
// `if (d <= span) atomicAdd(...)` is a divergent region per key with the shared window address re-derived inside
// (13 instructions per key instead of 6).  hist_s: shared-window address of the histogram.
#define BG_HIST_SPARE 268
__device__ __forceinline__ void bg_hist_add(unsigned hist_s, unsigned d, unsigned span, int sh) {
    const unsigned bin = (d <= span) ? (d >> sh) : (unsigned)BG_HIST_SPARE;
    asm volatile("red.shared.add.u32 [%0], 1;" :: "r"(hist_s + (bin << 2)) : "memory");
}

// the scalar path of bg_load4 (ragged cells, unaligned frames): out of line, it is rare and sixteen inlined copies of it
// spread the hot path of bg_cells_kernel over the instruction cache
template <bool FUSED>
__device__ __noinline__ float bg_load_slow(const FrameArgs f, int W, int H, int x, int y) { return load_px<FUSED>(f, W, H, x, y); }

// Four consecutive pixels starting at (x, y), x % 4 == 0: calibrated value, NaN where masked / outside [0, x_end).
template <bool FUSED>
__device__ __forceinline__ void bg_load4(const FrameArgs& f, int W, int H, int x, int y, int x_end, float v[4]) {
    if (y >= H || x >= x_end) { v[0] = v[1] = v[2] = v[3] = nanf_(); return; }
    if (f.vec_ok && x + 3 < x_end) {
        size_t o = (size_t)y * W + x;
        if (FUSED && f.pre) {
            const float4 c = calib4_pre<false>(f, o);
            v[0] = c.x; v[1] = c.y; v[2] = c.z; v[3] = c.w;
        } else if (FUSED) {
            uint2 rw = __ldg(reinterpret_cast<const uint2*>(f.raw + o));
            float4 b = __ldg(reinterpret_cast<const float4*>(f.bias + o));
            float4 d = __ldg(reinterpret_cast<const float4*>(f.dark + o));
            float4 fl = __ldg(reinterpret_cast<const float4*>(f.flat + o));
            unsigned bp = f.bpm ? __ldg(reinterpret_cast<const unsigned*>(f.bpm + o)) : 0u;
#ifndef BG_SCALAR_CALIB
            // four pixels in packed FP32 with the all-good fast path (calib_fast4: the values calib_px gives for normal flats)
            int bad4 = 0;
            const unsigned fmin_bits = __float_as_uint(f.flat_min);
            const float4 c = calib_fast4<false>(rw, b, d, fl, f.t_exp, (float)f.sat_adu, fmin_bits, 0x7f800000u - fmin_bits, bad4);
            v[0] = c.x; v[1] = c.y; v[2] = c.z; v[3] = c.w;
            if (bp) {
                if (bp & 0xffu) v[0] = nanf_();
                if (bp & 0xff00u) v[1] = nanf_();
                if (bp & 0xff0000u) v[2] = nanf_();
                if (bp & 0xff000000u) v[3] = nanf_();
            }
#else
            int r0 = rw.x & 0xffff, r1 = rw.x >> 16, r2 = rw.y & 0xffff, r3 = rw.y >> 16;
            v[0] = calib_px((float)r0, b.x, d.x, fl.x, r0 >= f.sat_adu || (bp & 0xffu), f.t_exp, f.flat_min);
            v[1] = calib_px((float)r1, b.y, d.y, fl.y, r1 >= f.sat_adu || (bp & 0xff00u), f.t_exp, f.flat_min);
            v[2] = calib_px((float)r2, b.z, d.z, fl.z, r2 >= f.sat_adu || (bp & 0xff0000u), f.t_exp, f.flat_min);
            v[3] = calib_px((float)r3, b.w, d.w, fl.w, r3 >= f.sat_adu || (bp & 0xff000000u), f.t_exp, f.flat_min);
#endif
        } else {
            float4 c = __ldg(reinterpret_cast<const float4*>(f.cal + o));
            unsigned m = __ldg(reinterpret_cast<const unsigned*>(f.mask + o));
            v[0] = (m & 0xffu) ? c.x : nanf_();
            v[1] = (m & 0xff00u) ? c.y : nanf_();
            v[2] = (m & 0xff0000u) ? c.z : nanf_();
            v[3] = (m & 0xff000000u) ? c.w : nanf_();
        }
    } else {
#pragma unroll
        for (int i = 0; i < 4; ++i) v[i] = (x + i < x_end) ? bg_load_slow<FUSED>(f, W, H, x + i, y) : nanf_();
    }
}

// CTA-wide sum of one int per thread.  s_red[16..18] are three rotating counters (zero at kernel start): call n adds
// into counter n mod 3 and clears counter (n + 1) mod 3, whose last readers passed the previous barrier; `it` is the
// caller's rotating index.  One warp reduction, one shared atomic per warp, one barrier, one load.
__device__ __forceinline__ int bg_block_sum(int v, int* s_red, int& par, int& it) {
    (void)par;
    v = __reduce_add_sync(0xffffffffu, v);
    int* ctr = s_red + 16;
    const int nxt = it == 2 ? 0 : it + 1;
    if ((threadIdx.x & 31) == 0) atomicAdd(ctr + it, v);
    if (threadIdx.x == 32) ctr[nxt] = 0;
    __syncthreads();
    const int r = ctr[it];
    it = nxt;
    return r;
}
__device__ __forceinline__ unsigned bg_block_min(unsigned v, int* s_red, int& par) {
    v = __reduce_min_sync(0xffffffffu, v);
    unsigned* r = reinterpret_cast<unsigned*>(s_red + par * 8);
    if ((threadIdx.x & 31) == 0) r[threadIdx.x >> 5] = v;
    __syncthreads();
    uint4 a = *reinterpret_cast<const uint4*>(r), b = *reinterpret_cast<const uint4*>(r + 4);
    par ^= 1;
    return min(min(min(a.x, a.y), min(a.z, a.w)), min(min(b.x, b.y), min(b.z, b.w)));
}
__device__ __forceinline__ unsigned bg_block_max_valid(unsigned v, int* s_red, int& par) {   // v = 0 for "none"
    v = __reduce_max_sync(0xffffffffu, v);
    unsigned* r = reinterpret_cast<unsigned*>(s_red + par * 8);
    if ((threadIdx.x & 31) == 0) r[threadIdx.x >> 5] = v;
    __syncthreads();
    uint4 a = *reinterpret_cast<const uint4*>(r), b = *reinterpret_cast<const uint4*>(r + 4);
    par ^= 1;
    return max(max(max(a.x, a.y), max(a.z, a.w)), max(max(b.x, b.y), max(b.z, b.w)));
}

// k-th smallest (0-based, k < n) of the n non-sentinel keys held by the CTA (BG_KPT per thread).
// Multi-level counting select: the live key range [lo, hi] is cut into <= 256 equal bins (width a power of two), the keys
// inside it are counted into a shared histogram, a CTA-wide scan finds the bin that holds rank k, and that bin becomes the
// new range -- 8 bits per level.  Once <= BG_FINISH keys remain they are ranked directly in one warp.  Exact.
// The first range is either [kmin, kmax], the extremes of the keys (GUESS = false: c_lo = 0, cnt = n), or a GUESS from a
// sample (bg_sample_range): then the first level also counts the keys below the range, and the call returns false, with
// nothing selected, when rank k lies outside it (the caller falls back to the extremes).
// s_hist: 256 + 12 + 4 words, s_list: BG_FINISH + 2 words, s_cnt: 1 word of shared memory.
__device__ __forceinline__ bool bg_select(const bool GUESS, const unsigned (&key)[BG_KPT], int k, int n, unsigned lo, unsigned hi,
                                          int* s_hist, unsigned* s_list, int* s_cnt, unsigned& kth, unsigned& next, bool& have_next) {
    int c_lo = 0, cnt = n;                          // #{key < lo}, #{lo <= key <= hi}
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    int* s_w = s_hist + 256;                        // [0..7] warp totals, [8..10] picked bin, its prefix, its count, [11] keys below
    bool first = GUESS;
    if (GUESS) __syncthreads();                     // s_w[8..11] of the previous select are still being read
    while (first || (cnt > BG_FINISH && hi > lo)) {
        const int sh = max(0, 24 - __clz(hi - lo)); // (hi - lo) >> sh <= 255
        s_hist[tid] = 0;
        if (first && tid < 4) s_w[8 + tid] = (tid == 0) ? -1 : 0;
        __syncthreads();
        const unsigned span = hi - lo, hist_s = (unsigned)__cvta_generic_to_shared(s_hist);
        int below = 0;
#pragma unroll
        for (int i = 0; i < BG_KPT; ++i) {
            const unsigned d = key[i] - lo;             // wraps to a huge value below lo: one compare covers both ends
            bg_hist_add(hist_s, d, span, sh);
            if (GUESS) below += (key[i] < lo) ? 1 : 0;
        }
        if (first) {
            below = __reduce_add_sync(0xffffffffu, below);
            if (lane == 0 && below) atomicAdd(s_w + 11, below);
        }
        __syncthreads();
        const int h = s_hist[tid];
        int inc = h;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const int o = __shfl_up_sync(0xffffffffu, inc, d);
            if (lane >= d) inc += o;
        }
        if (lane == 31) s_w[wid] = inc;
        __syncthreads();
#pragma unroll
        for (int w = 0; w < 7; ++w) inc += (w < wid) ? s_w[w] : 0;
        if (first) c_lo = s_w[11];
        const int krel = k - c_lo;
        if (inc - h <= krel && krel < inc) { s_w[8] = tid; s_w[9] = inc - h; s_w[10] = h; }
        __syncthreads();
        if (first && s_w[8] < 0) return false;        // rank k is not in the guessed range (uniform: every thread reads s_w[8])
        first = false;
        const unsigned bin = (unsigned)s_w[8];
        c_lo += s_w[9];
        cnt = s_w[10];
        lo += bin << sh;
        const unsigned top = lo + ((1u << sh) - 1u);
        hi = (top < lo) ? hi : min(hi, top);          // top < lo: wrapped past 2^32
    }
    // `next` = the key of rank k + 1 when it lies in the same final range (have_next), for the even-n median
    if (hi == lo) { have_next = (k - c_lo + 1 < cnt); next = lo; kth = lo; return true; }
    // at most BG_FINISH keys remain in [lo, hi]: rank them directly (ties by list position)
    if (tid == 0) *s_cnt = 0;
    __syncthreads();
#pragma unroll
    for (int i = 0; i < BG_KPT; ++i)
        if (key[i] >= lo && key[i] <= hi) {
            int p = atomicAdd(s_cnt, 1);
            if (p < BG_FINISH) s_list[p] = key[i];
        }
    __syncthreads();
    const int m = min(*s_cnt, BG_FINISH);           // read by every thread before the last barrier of this call
    if (tid < 32) {
        const unsigned mine = (lane < m) ? s_list[lane] : BG_SENTINEL;
        int rank = 0;
        for (int j = 0; j < m; ++j) {
            unsigned kj = __shfl_sync(0xffffffffu, mine, j);
            rank += (kj < mine || (kj == mine && j < lane)) ? 1 : 0;
        }
        if (lane < m && rank == k - c_lo) s_list[BG_FINISH] = mine;
        if (lane < m && rank == k - c_lo + 1) s_list[BG_FINISH + 1] = mine;
    }
    __syncthreads();
    have_next = (k - c_lo + 1 < m);
    next = s_list[BG_FINISH + 1];
    kth = s_list[BG_FINISH];
    return true;
}

// median rule of R-D1: (v_((n-1)/2) + v_(n/2)) / 2 as keys -> the two central keys.  [glo, ghi] (glo <= ghi): a guess of a
// range that holds them (bg_sample_range); when it does not, or there is none (glo > ghi), the select starts from the
// extremes of the keys, which are then found first.
__device__ __forceinline__ void bg_central_pair(const unsigned (&key)[BG_KPT], int n, unsigned glo, unsigned ghi, int* s_red,
                                                int& par, int& it, int* s_hist, unsigned* s_list, int* s_cnt, unsigned& k1,
                                                unsigned& k2) {
    const int r = (n - 1) >> 1;
    unsigned nxt_sel;
    bool have_next;
    // one copy of the select in the instruction stream (the kernel is instruction-fetch bound otherwise): a failed guess
    // comes round again from the extremes
    bool guess = glo <= ghi;
#pragma unroll 1
    for (;;) {
        if (!guess) {
            unsigned lo = BG_SENTINEL, hi = 0u;
#pragma unroll
            for (int i = 0; i < BG_KPT; ++i) {
                lo = min(lo, key[i]);
                hi = max(hi, key[i] != BG_SENTINEL ? key[i] : 0u);
            }
            glo = bg_block_min(lo, s_red, par);
            ghi = bg_block_max_valid(hi, s_red, par);
        }
        if (bg_select(guess, key, r, n, glo, ghi, s_hist, s_list, s_cnt, k1, nxt_sel, have_next)) break;
        guess = false;
    }
    k2 = k1;
    if ((n & 1) == 0) {
        if (have_next) {                            // rank r + 1 fell into the same final range (the usual case)
            k2 = nxt_sel;
        } else {                                    // k1 again if it repeats, else the next larger key
            int c = 0;
            unsigned nxt = BG_SENTINEL;
#pragma unroll
            for (int i = 0; i < BG_KPT; ++i) {
                c += (key[i] <= k1) ? 1 : 0;
                if (key[i] > k1) nxt = min(nxt, key[i]);
            }
            c = bg_block_sum(c, s_red, par, it);
            nxt = bg_block_min(nxt, s_red, par);
            if (r + 1 >= c) k2 = nxt;
        }
    }
}

// Sample quartiles: 64 of the cell's keys (one of every fourth thread) are ranked by two warps; q[0..2] = the sample's quartile keys, q[3] = number of valid samples (all threads).  They only steer
// where the exact select starts.
__device__ __forceinline__ void bg_sample_quartiles(const unsigned (&key)[BG_KPT], unsigned* s_samp, unsigned (&q)[4]) {
    const int tid = threadIdx.x;
    if ((tid & 3) == 0) {                           // column group c of the cell, row block c: a diagonal of 16 x 4 pixels
        const int j = (tid >> 2) & 3;
        s_samp[tid >> 2] = j == 0 ? key[1] : j == 1 ? key[5] : j == 2 ? key[9] : key[13];
    }
    if (tid < 4) s_samp[64 + tid] = 0u;
    __syncthreads();
    if (tid < 64) {
        const unsigned mine = s_samp[tid];
        int rank = 0, nv = 0;
#pragma unroll
        for (int j = 0; j < 64; j += 4) {
            const uint4 o = *reinterpret_cast<const uint4*>(s_samp + j);
            rank += (o.x < mine || (o.x == mine && j < tid)) + (o.y < mine || (o.y == mine && j + 1 < tid)) +
                    (o.z < mine || (o.z == mine && j + 2 < tid)) + (o.w < mine || (o.w == mine && j + 3 < tid));
            nv += (o.x != BG_SENTINEL) + (o.y != BG_SENTINEL) + (o.z != BG_SENTINEL) + (o.w != BG_SENTINEL);
        }
        if (rank == nv >> 2) s_samp[64] = mine;
        if (rank == nv >> 1) s_samp[65] = mine;
        if (rank == (3 * nv) >> 2) s_samp[66] = mine;
        if (tid == 0) s_samp[67] = (unsigned)nv;
    }
    __syncthreads();
    q[0] = s_samp[64]; q[1] = s_samp[65]; q[2] = s_samp[66]; q[3] = s_samp[67];
}

// Detection candidates of argus_detect_frame ("one pass"): while a cell's pixels are in registers,
// bg_cells_kernel<., true> notes every good pixel with |v - med| > kappa * sig (all good pixels of an invalid cell) in the
// cell's own candidate list and stores cut = med + kappa * sig per cell (-inf: invalid cell).  det_cand_kernel later proves
// per 64 x 32-pixel detection tile that no pixel below its cells' cuts can pass the detection threshold and then looks at
// the candidates of the cells it overlaps only; tiles where the proof fails or a list overflowed are scanned in full.
// Lists are per cell, so bg_cells_kernel writes them with plain stores (no global atomic, nothing to clear): a cell of
// B <= 32 lies in one tile (one list of det_cand_cap(B) entries); a cell of 64 is two stacked tiles (two lists).
#define DET_TW 64
#define DET_TH 32
#define DET_CAND_CAP 48              // candidates looked at per tile (2.3 % of its pixels); more: the tile is scanned in full
__host__ __device__ __forceinline__ int det_cand_cap(int B) { return B == 64 ? DET_CAND_CAP : B == 32 ? 24 : B == 16 ? 8 : 4; }
struct BgCand {
    unsigned* cnt;                   // [n_lists] candidates found per list (may exceed its capacity); n_lists = G (2 G at B = 64)
    unsigned short* list;            // [n_lists][det_cand_cap(B)] position in the tile: (y - y0) * 64 + (x - x0)
    float* cut;                      // [G]
    float kappa;
};

struct BgCandShared {
    unsigned short loc[2][DET_CAND_CAP];
    unsigned n[2];
};
__device__ __forceinline__ void bg_cand_push(BgCandShared& sc, int x0, int y0, int lx, int ly, int B) {
    const int h = (B == 64) ? (ly >> 5) : 0;
    const unsigned pos = atomicAdd(&sc.n[h], 1u);
    if (pos < DET_CAND_CAP) sc.loc[h][pos] = (unsigned short)(((y0 + ly) % DET_TH) * DET_TW + (x0 + lx) % DET_TW);
}
// all threads of the CTA, after the last push
__device__ __forceinline__ void bg_cand_flush(BgCandShared& sc, const BgCand& cd, int cell, int B) {
    __syncthreads();
    const int tid = threadIdx.x, h = tid >> 6, t = tid & 63, cap = det_cand_cap(B);
    if (h >= (B == 64 ? 2 : 1)) return;
    const size_t l = (B == 64) ? 2 * (size_t)cell + h : (size_t)cell;
    const unsigned n = sc.n[h];
    if (t == 0) cd.cnt[l] = n;
    if (t < min(n, (unsigned)cap)) cd.list[l * cap + t] = sc.loc[h][t];
}

// R-D1: per-cell median, 1.4826 MAD and good-pixel count.  grid = GX * GY CTAs of 256 threads; B in {8,16,32,64}.
#ifndef BG_MINB
#define BG_MINB 6                    // 40 registers, no spills: the kernel waits at its barriers, residency pays (4 / 5 CTAs per SM: 11 % / 2 % slower)
#endif
template <bool FUSED, bool CAND = false>
__global__ void __launch_bounds__(BG_THREADS, BG_MINB) bg_cells_kernel(FrameArgs f, int W, int H, int B, int GX, int n_min,
                                                              float* __restrict__ med_out, float* __restrict__ sig_out,
                                                              int* __restrict__ ngood_out, BgCand cd) {
    __shared__ __align__(16) int s_red[20];
    __shared__ unsigned s_list[BG_FINISH + 2];
    __shared__ int s_hist[256 + 12 + 4];
    __shared__ int s_cnt;
    __shared__ __align__(16) unsigned s_samp[68];
    __shared__ BgCandShared s_cand;
    if (threadIdx.x < 3) s_red[16 + threadIdx.x] = 0;
    if (CAND && threadIdx.x < 2) s_cand.n[threadIdx.x] = 0u;
    __syncthreads();
    const int cell = blockIdx.x, gx = cell % GX, gy = cell / GX;
    const int x0 = gx * B, y0 = gy * B, x_end = min(x0 + B, W), y_end = min(y0 + B, H);
    const int col = (threadIdx.x & 15) * 4, row = threadIdx.x >> 4;
    unsigned key[BG_KPT];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        float v[4];
        bg_load4<FUSED>(f, W, y_end, x0 + col, y0 + row + 16 * j, x_end, v);
#pragma unroll
        for (int i = 0; i < 4; ++i) key[4 * j + i] = bg_key(v[i]);
    }
    int par = 0, it = 0;
    int n = 0;
#pragma unroll
    for (int i = 0; i < BG_KPT; ++i) n += (key[i] != BG_SENTINEL) ? 1 : 0;
    n = bg_block_sum(n, s_red, par, it);
    if (n < max(n_min, 1)) {
        if (threadIdx.x == 0) { med_out[cell] = 0.f; sig_out[cell] = 0.f; ngood_out[cell] = n; }
        if (CAND) {                                  // no statistics to cut on: every good pixel is a candidate
            if (threadIdx.x == 0) cd.cut[cell] = __int_as_float(0xff800000);
            unsigned m = 0u;
#pragma unroll
            for (int i = 0; i < BG_KPT; ++i) m |= (key[i] != BG_SENTINEL) ? (1u << i) : 0u;
            while (m) {
                const int i = __ffs(m) - 1;
                m &= m - 1u;
                bg_cand_push(s_cand, x0, y0, col + (i & 3), row + 16 * (i >> 2), B);
            }
            bg_cand_flush(s_cand, cd, cell, B);
        }
        return;
    }
    // where the selects start: [median - sigma, median + sigma] and 1.4826 MAD in [0.35, 1.35] sigma of a 64-key sample
    // (the exact selects fall back to the extremes of the keys when the rank is not in there)
    unsigned q[4];
    bg_sample_quartiles(key, s_samp, q);
    unsigned glo = 1u, ghi = 0u, dlo = 1u, dhi = 0u;  // lo > hi: no guess
    if (q[3] >= BG_SAMPLE_MIN) {
        const float m0 = bg_unkey(q[1]), s0 = 0.7413f * (bg_unkey(q[2]) - bg_unkey(q[0]));
        if (s0 >= 0.f && s0 < __int_as_float(0x7f800000)) {
            glo = bg_key(m0 - s0); ghi = bg_key(m0 + s0);
            dlo = __float_as_uint(0.35f * 0.6745f * s0); dhi = __float_as_uint(1.35f * 0.6745f * s0);
        }
    }
    unsigned k1, k2;
    float med = 0.f;
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {           // median of the values, then of |v - med| (one copy of the code)
        bg_central_pair(key, n, pass ? dlo : glo, pass ? dhi : ghi, s_red, par, it, s_hist, s_list, &s_cnt, k1, k2);
        if (pass == 0) {
            med = 0.5f * (bg_unkey(k1) + bg_unkey(k2));
            // MAD: |v - med| >= 0, whose bit patterns are already ordered
#pragma unroll
            for (int i = 0; i < BG_KPT; ++i)
                key[i] = (key[i] != BG_SENTINEL) ? __float_as_uint(fabsf(bg_unkey(key[i]) - med)) : BG_SENTINEL;
        }
    }
    const float mad = 0.5f * (__uint_as_float(k1) + __uint_as_float(k2));
    if (threadIdx.x == 0) { med_out[cell] = med; sig_out[cell] = BG_MAD_TO_SIGMA * mad; ngood_out[cell] = n; }
    if (CAND) {
        const float cthr = cd.kappa * (BG_MAD_TO_SIGMA * mad);
        if (threadIdx.x == 0) cd.cut[cell] = med + cthr;
        unsigned m = 0u;                             // the sentinel reads as NaN: never above the cut
#pragma unroll
        for (int i = 0; i < BG_KPT; ++i) m |= (__uint_as_float(key[i]) > cthr) ? (1u << i) : 0u;
        while (m) {                                  // 0.9 % of the pixels: one or two rounds per warp
            const int i = __ffs(m) - 1;
            m &= m - 1u;
            bg_cand_push(s_cand, x0, y0, col + (i & 3), row + 16 * (i >> 2), B);
        }
        bg_cand_flush(s_cand, cd, cell, B);
    }
}

// R-D2: 3x3 median over the valid cells (clipped to the grid); no valid cell: bkg = 0, nse = +inf.
__device__ __forceinline__ float bg_median_small(float* v, int m) {
    for (int i = 1; i < m; ++i) {
        float x = v[i];
        int j = i - 1;
        while (j >= 0 && v[j] > x) { v[j + 1] = v[j]; --j; }
        v[j + 1] = x;
    }
    return 0.5f * (v[(m - 1) >> 1] + v[m >> 1]);
}
__global__ void __launch_bounds__(128) bg_filter_kernel(const float* __restrict__ med, const float* __restrict__ sig,
                                                        const int* __restrict__ ngood, int GX, int GY, int n_min,
                                                        float* __restrict__ bkg, float* __restrict__ nse) {
    const int c = blockIdx.x * 128 + threadIdx.x;
    if (c >= GX * GY) return;
    const int gx = c % GX, gy = c / GX;
    float a[9], b[9];
    int m = 0;
    for (int y = max(gy - 1, 0); y <= min(gy + 1, GY - 1); ++y)
        for (int x = max(gx - 1, 0); x <= min(gx + 1, GX - 1); ++x) {
            const int q = y * GX + x;
            if (ngood[q] >= max(n_min, 1)) { a[m] = med[q]; b[m] = sig[q]; ++m; }
        }
    bkg[c] = m ? bg_median_small(a, m) : 0.f;
    nse[c] = m ? bg_median_small(b, m) : __int_as_float(0x7f800000);
}

// ------------------------------------------------------------------------------------------------ detection
#define DET_PITCH 66                 // 64 + 2 apron columns; 66 mod 32 = 2 spreads a warp's four rows over the banks
#define DET_PCOLS 12                 // node columns a tile can touch: (DET_TW + 2) / 8 + 2 at B = 8

struct DetGrid {
    const float* bkg;
    const float* nse;
    int B, GX, GY;
    float inv_B, half;               // 1 / B, (B - 1) / 2
    float k_sigma;
};

// R-D3 along one axis: lower node and fraction of pixel coordinate p (clamped outside the outermost centres).
__device__ __forceinline__ void det_node(int p, const DetGrid& g, int G, int& g0, float& t) {
    const float u = fminf(fmaxf(((float)p - g.half) * g.inv_B, 0.f), (float)(G - 1));
    g0 = min((int)u, max(G - 2, 0));
    t = u - (float)g0;
}
// R-D4 / R-D5 on one 64 x 32 tile.  tile_info[tile] = (base of the tile's records in tmp, count); *total counts all.
// Staging: the grids are interpolated along y once per tile row (s_rb / s_rn, straight from the L2-resident grids), the
// x node and fraction of every tile column are tabulated (s_col): a pixel's background costs two shared loads + one FMA.
// R-D5 record of the source at (x, y): q = s over its 3 x 3 window in raster order (-inf: masked or off-frame), bkg / nse the
// interpolated maps at the peak.  One function for both detection paths (their catalogues are identical bit for bit).
__device__ __forceinline__ void det_write_record(ArgusSourceRec* __restrict__ dst_rec, int x, int y, const float (&q)[9], float bkg,
                                                 float nse) {
    const float ninf = __int_as_float(0xff800000);
    float flux = 0.f, mx = 0.f, my = 0.f;
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const float v = q[3 * r + c];
            if (v != ninf) { flux += v; mx += v * (float)(c - 1); my += v * (float)(r - 1); }
        }
    const float cx = flux > 0.f ? mx / flux : 0.f, cy = flux > 0.f ? my / flux : 0.f;
    uint4* dst = reinterpret_cast<uint4*>(dst_rec);
    dst[0] = make_uint4((unsigned)x, (unsigned)y, __float_as_uint(q[4]), __float_as_uint(flux));
    dst[1] = make_uint4(__float_as_uint(cx), __float_as_uint(cy), __float_as_uint(bkg), __float_as_uint(nse));
}

template <bool FUSED>
__device__ __forceinline__ void det_tile_body(const int tile, const FrameArgs& f, int W, int H, const DetGrid& g, int tiles_x,
                                              ArgusSourceRec* __restrict__ tmp, unsigned capacity,
                                              uint2* __restrict__ tile_info, unsigned* __restrict__ total,
                                              unsigned* __restrict__ band_cnt) {
    __shared__ float s_s[(DET_TH + 2) * DET_PITCH];
    __shared__ float s_rb[DET_TH + 2][DET_PCOLS], s_rn[DET_TH + 2][DET_PCOLS];
    __shared__ float2 s_col[DET_PITCH];              // (.x: node offsets lx | lx1 << 8 as int bits, .y: tx)
    __shared__ int s_warp[8];
    __shared__ unsigned s_base, s_nmin;              // s_nmin: bits of the smallest noise node the tile touches
    if (threadIdx.x == 0) s_nmin = 0x7f800000u;
    __syncthreads();
    const int x0 = (tile % tiles_x) * DET_TW, y0 = (tile / tiles_x) * DET_TH, tid = threadIdx.x;
    int pgx;
    float tdummy;
    det_node(x0 - 1, g, g.GX, pgx, tdummy);
    // tables straight from the (L2-resident) grids: y-interpolated node rows and the per-column (node, fraction).
    // Only the node columns the tile touches are built (3 at cell 64, 11 at cell 8).
    int pgx1;
    det_node(x0 + DET_TW, g, g.GX, pgx1, tdummy);
    const int ncols = min(pgx1 + 1, g.GX - 1) - pgx + 1;
    const float inv_ncols = 1.0f / (float)ncols;
    float nmin = __int_as_float(0x7f800000);
    for (int e = tid; e < (DET_TH + 2) * ncols; e += 256) {
        const int r = (int)(((float)e + 0.5f) * inv_ncols), c = e - r * ncols;   // exact: e < 2^10, ncols <= 12
        int gy0;
        float ty;
        det_node(y0 - 1 + r, g, g.GY, gy0, ty);
        const int col = min(pgx + c, g.GX - 1), q0 = gy0 * g.GX + col, q1 = min(gy0 + 1, g.GY - 1) * g.GX + col;
        const float b0 = __ldg(g.bkg + q0), b1 = __ldg(g.bkg + q1), n0 = __ldg(g.nse + q0), n1 = __ldg(g.nse + q1);
        s_rb[r][c] = fmaf(ty, b1 - b0, b0);
        s_rn[r][c] = fmaf(ty, n1 - n0, n0);
        nmin = fminf(nmin, fminf(n0, n1));
    }
    {   // noise nodes are >= 0 or +inf: their bit patterns order like the values
        const unsigned m = __reduce_min_sync(0xffffffffu, __float_as_uint(nmin));
        if ((tid & 31) == 0 && m != 0x7f800000u) atomicMin(&s_nmin, m);
    }
    if (tid >= 128 && tid < 128 + DET_PITCH) {
        int gx0;
        float tx;
        det_node(x0 - 1 + (tid - 128), g, g.GX, gx0, tx);
        s_col[tid - 128] = make_float2(__int_as_float((gx0 - pgx) | ((min(gx0 + 1, g.GX - 1) - pgx) << 8)), tx);
    }
    __syncthreads();
    const float ninf = __int_as_float(0xff800000);   // -inf: masked and off-frame pixels never win, never count
    // interior: (DET_TH + 2) rows x 16 groups of four pixels (vector loads); apron columns: one pixel each side
    for (int e = tid; e < (DET_TH + 2) * 16; e += 256) {
        const int r = e >> 4, q = e & 15, py = y0 - 1 + r;
        float v[4];
        if (py >= 0) bg_load4<FUSED>(f, W, H, x0 + 4 * q, py, W, v);
        else v[0] = v[1] = v[2] = v[3] = nanf_();
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int c = 1 + 4 * q + i;
            const float2 ci = s_col[c];
            const int lx = __float_as_int(ci.x) & 0xff, lx1 = __float_as_int(ci.x) >> 8;
            const float b0 = s_rb[r][lx];
            const float s = v[i] - fmaf(ci.y, s_rb[r][lx1] - b0, b0);
            s_s[r * DET_PITCH + c] = (v[i] == v[i]) ? s : ninf;
        }
    }
    if (tid < 2 * (DET_TH + 2)) {
        const int r = tid >> 1, c = (tid & 1) ? DET_PITCH - 1 : 0;
        const float v = load_px<FUSED>(f, W, H, x0 - 1 + c, y0 - 1 + r);
        const float2 ci = s_col[c];
        const int lx = __float_as_int(ci.x) & 0xff, lx1 = __float_as_int(ci.x) >> 8;
        const float b0 = s_rb[r][lx];
        s_s[r * DET_PITCH + c] = (v == v) ? v - fmaf(ci.y, s_rb[r][lx1] - b0, b0) : ninf;
    }
    __syncthreads();
    // each thread: 8 consecutive pixels of one row.  Threshold first: every interpolated noise value of the tile is a
    // convex combination of the nodes it touches, so s > k * (smallest node) is necessary -- one compare per pixel
    // rejects all but ~1e-3 of them; only the survivors look at their neighbours and at the exact threshold.
    const int ry = tid >> 3, cx0 = (tid & 7) * 8;
    const float thr_min = 0.999999f * (g.k_sigma * __uint_as_float(s_nmin));   // slack for the rounding of the lerp
    const float* row = s_s + (ry + 1) * DET_PITCH + cx0 + 1;
    unsigned bits = 0;
    const int py = y0 + ry;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        const float c = row[j];
        if (c > thr_min && c > 0.f) {                    // false for -inf (masked, off-frame) and for thr_min NaN
            const float* q = row + j;
            const float e4 = fmaxf(fmaxf(q[-DET_PITCH - 1], q[-DET_PITCH]), fmaxf(q[-DET_PITCH + 1], q[-1]));
            const float l4 = fmaxf(fmaxf(q[1], q[DET_PITCH - 1]), fmaxf(q[DET_PITCH], q[DET_PITCH + 1]));
            if (c > e4 && c >= l4) {                     // raster-first pixel wins ties
                const float2 ci = s_col[cx0 + j + 1];
                const int lx = __float_as_int(ci.x) & 0xff, lx1 = __float_as_int(ci.x) >> 8;
                const float n0 = s_rn[ry + 1][lx];
                const float nse = fmaf(ci.y, s_rn[ry + 1][lx1] - n0, n0);
                if (c > g.k_sigma * nse) bits |= 1u << j;   // false for nse = +inf or NaN (undefined background)
            }
        }
    }
    // CTA-wide exclusive scan of the per-thread counts (thread order = raster order inside the tile)
    const int cnt = __popc(bits), lane = tid & 31, wid = tid >> 5;
    int inc = cnt;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        int o = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += o;
    }
    if (lane == 31) s_warp[wid] = inc;
    __syncthreads();
    int before = inc - cnt, tile_cnt = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const int c = s_warp[k];
        before += (k < wid) ? c : 0;
        tile_cnt += c;
    }
    if (tid == 0) {
        const unsigned base = tile_cnt ? atomicAdd(total, (unsigned)tile_cnt) : 0u;
        if (tile_cnt) atomicAdd(band_cnt + tile / tiles_x, (unsigned)tile_cnt);
        tile_info[tile] = make_uint2(base, (unsigned)tile_cnt);
        s_base = base;
    }
    if (tile_cnt == 0) return;
    __syncthreads();
    unsigned pos = s_base + (unsigned)before;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        if (!((bits >> j) & 1u)) continue;
        float q[9];
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int c = 0; c < 3; ++c) q[3 * r + c] = row[j + (r - 1) * DET_PITCH + (c - 1)];
        const float2 ci = s_col[cx0 + j + 1];
        const int lx = __float_as_int(ci.x) & 0xff, lx1 = __float_as_int(ci.x) >> 8;
        const float b0 = s_rb[ry + 1][lx], n0 = s_rn[ry + 1][lx];
        if (pos < capacity)
            det_write_record(tmp + pos, x0 + cx0 + j, py, q, fmaf(ci.y, s_rb[ry + 1][lx1] - b0, b0),
                             fmaf(ci.y, s_rn[ry + 1][lx1] - n0, n0));
        ++pos;
    }
}

template <bool FUSED>
__global__ void __launch_bounds__(256, 8) det_tiles_kernel(FrameArgs f, int W, int H, DetGrid g, int tiles_x,
                                                           ArgusSourceRec* __restrict__ tmp, unsigned capacity,
                                                           uint2* __restrict__ tile_info, unsigned* __restrict__ total,
                                                           unsigned* __restrict__ band_cnt) {
    det_tile_body<FUSED>((int)blockIdx.x, f, W, H, g, tiles_x, tmp, capacity, tile_info, total, band_cnt);
}

// The same on a list of tiles (the tiles det_cand_kernel hands over): CTAs stride over list[0 .. *n_list).
template <bool FUSED>
__global__ void __launch_bounds__(256, 8) det_tiles_list_kernel(FrameArgs f, int W, int H, DetGrid g, int tiles_x,
                                                                ArgusSourceRec* __restrict__ tmp, unsigned capacity,
                                                                uint2* __restrict__ tile_info, unsigned* __restrict__ total,
                                                                unsigned* __restrict__ band_cnt,
                                                                const unsigned* __restrict__ list, const unsigned* __restrict__ n_list) {
    const unsigned n = *n_list;
    for (unsigned i = blockIdx.x; i < n; i += gridDim.x) {
        __syncthreads();                              // the previous tile's shared tables are still being read
        det_tile_body<FUSED>((int)list[i], f, W, H, g, tiles_x, tmp, capacity, tile_info, total, band_cnt);
    }
}

// ---- candidate path of argus_detect_frame.  s and the maps at one pixel, with the arithmetic of det_tile_body: the grids are
// interpolated along y first (fmaf(ty, b1 - b0, b0) per node column), then along x.
struct DetAt {
    int q00, q01, q10, q11;
    float tx, ty;
};
__device__ __forceinline__ DetAt det_at(const DetGrid& g, int x, int y) {
    DetAt a;
    int gx0, gy0;
    det_node(x, g, g.GX, gx0, a.tx);
    det_node(y, g, g.GY, gy0, a.ty);
    const int c1 = min(gx0 + 1, g.GX - 1), r1 = min(gy0 + 1, g.GY - 1);
    a.q00 = gy0 * g.GX + gx0; a.q01 = gy0 * g.GX + c1; a.q10 = r1 * g.GX + gx0; a.q11 = r1 * g.GX + c1;
    return a;
}
__device__ __forceinline__ float det_lerp(const float* __restrict__ grid, const DetAt& a) {
    const float v00 = __ldg(grid + a.q00), v01 = __ldg(grid + a.q01), v10 = __ldg(grid + a.q10), v11 = __ldg(grid + a.q11);
    const float r0 = fmaf(a.ty, v10 - v00, v00), r1 = fmaf(a.ty, v11 - v01, v01);
    return fmaf(a.tx, r1 - r0, r0);
}
// MODE 0: cal + mask, 1: raw + masters, 2: raw + pre-fused masters.  Pixel at element offset o (clamped into the frame by
// the caller, `in` = the pixel lies in the frame): no branch on the data, so that the loads of a 3 x 3 window are issued
// together; the values are those of load_px.
template <int MODE>
__device__ __forceinline__ float det_px(const FrameArgs& f, size_t o, bool in) {
    float v;
    if (MODE == 2) {
        const int r = f.raw[o];
        v = calib_pre<false>((float)r, pre_load(f.offset, o, f.pre), pre_load(f.gain, o, f.pre), r >= f.sat_adu);
    } else if (MODE == 1) {
        const int r = f.raw[o];
        const float b = f.bias[o], d = f.dark[o], fl = f.flat[o];
        const bool bad = (r >= f.sat_adu) || (f.bpm && f.bpm[o] != 0);
        v = calib_px((float)r, b, d, fl, bad, f.t_exp, f.flat_min);
    } else {
        const float c = f.cal[o];
        v = f.mask[o] ? c : nanf_();
    }
    return in ? v : nanf_();
}

// One tile's candidates in one warp: R-D4 with the decisions of det_tile_body (threshold, then the 8 neighbours), records of
// the sources staged in shared memory (rec: DET_CAND_CAP x 2 uint4 of this warp).  Returns the lane's flags: bit it = its
// candidate it * 32 + lane is a source.  The node and fraction of the three columns and rows of the window are formed once.
template <int MODE>
__device__ __forceinline__ unsigned det_cand_tile(const FrameArgs& f, int W, int H, const DetGrid& g, int x0, int y0, unsigned cnt,
                                                  const unsigned short* mine, uint4* rec, int lane) {
    const float ninf = __int_as_float(0xff800000);
    unsigned flags = 0;
    for (unsigned it = 0; it * 32 < cnt; ++it) {
        const unsigned i = it * 32 + lane;
        if (i >= cnt) break;
        const int loc = mine[i], x = x0 + (loc & (DET_TW - 1)), y = y0 + (loc >> 6);
        int gx0[3], gx1[3], gy0[3], gy1[3], xs[3];
        float tx[3], ty[3];
        size_t ro[3];
        bool inx[3], iny[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const int xx = x + k - 1, yy = y + k - 1, yc = min(max(yy, 0), H - 1);
            inx[k] = (unsigned)xx < (unsigned)W; iny[k] = (unsigned)yy < (unsigned)H;
            xs[k] = min(max(xx, 0), W - 1);
            det_node(xs[k], g, g.GX, gx0[k], tx[k]);
            det_node(yc, g, g.GY, gy0[k], ty[k]);
            gx1[k] = min(gx0[k] + 1, g.GX - 1);
            gy1[k] = min(gy0[k] + 1, g.GY - 1) * g.GX;
            gy0[k] *= g.GX;
            ro[k] = (size_t)yc * W;
        }
        DetAt a;
        a.q00 = gy0[1] + gx0[1]; a.q01 = gy0[1] + gx1[1]; a.q10 = gy1[1] + gx0[1]; a.q11 = gy1[1] + gx1[1];
        a.tx = tx[1]; a.ty = ty[1];
        const float v = det_px<MODE>(f, ro[1] + xs[1], true);
        const float bkg = det_lerp(g.bkg, a), nse = det_lerp(g.nse, a);
        const float c = (v == v) ? v - bkg : ninf;
        if (!(c > 0.f && c > g.k_sigma * nse)) continue;   // false for nse = +inf or NaN (undefined background)
        float q[9];
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) {
                if (r == 1 && cc == 1) { q[4] = c; continue; }
                DetAt b;
                b.q00 = gy0[r] + gx0[cc]; b.q01 = gy0[r] + gx1[cc]; b.q10 = gy1[r] + gx0[cc]; b.q11 = gy1[r] + gx1[cc];
                b.tx = tx[cc]; b.ty = ty[r];
                const float vn = det_px<MODE>(f, ro[r] + xs[cc], inx[cc] && iny[r]);
                const float sn = vn - det_lerp(g.bkg, b);
                q[3 * r + cc] = (vn == vn) ? sn : ninf;
            }
        const float e4 = fmaxf(fmaxf(q[0], q[1]), fmaxf(q[2], q[3])), l4 = fmaxf(fmaxf(q[5], q[6]), fmaxf(q[7], q[8]));
        if (c > e4 && c >= l4) {                          // raster-first pixel wins ties
            flags |= 1u << it;
            det_write_record(reinterpret_cast<ArgusSourceRec*>(rec + 2 * i), x, y, q, bkg, nse);
        }
    }
    return flags;
}

// One warp per tile.  (1) Proof that the candidates are complete: every threshold bkg(p) + k nse(p) in the tile is a convex
// combination of bkg_g + k nse_g over the nodes g the tile touches, so a pixel that passes has v >= L - rounding with
// L = min_g (bkg_g + k nse_g); if L - slack >= max cut over the cells the tile overlaps, every such pixel was recorded by
// bg_cells_kernel (v > cut).  Otherwise, or when the list overflowed, the tile goes to fb_list (det_tiles_list_kernel).
// (2) R-D4 on the candidates with the decisions of det_tile_body (threshold, then the 8 neighbours), (3) records.
#ifndef DET_CAND_MINB
#define DET_CAND_MINB 4
#endif
template <bool FUSED>
__global__ void __launch_bounds__(256, DET_CAND_MINB) det_cand_kernel(FrameArgs f, int W, int H, DetGrid g, int tiles_x, int n_tiles,
                                                       const unsigned* __restrict__ cand_cnt,
                                                       const unsigned short* __restrict__ cand_list, const float* __restrict__ cut,
                                                       ArgusSourceRec* __restrict__ tmp, unsigned capacity,
                                                       uint2* __restrict__ tile_info, unsigned* __restrict__ total,
                                                       unsigned* __restrict__ band_cnt,
                                                       unsigned* __restrict__ fb_list, unsigned* __restrict__ fb_count) {
    const int lane = threadIdx.x & 31, tile = blockIdx.x * 8 + (threadIdx.x >> 5);
    if (tile >= n_tiles) return;
    const float inf = __int_as_float(0x7f800000);
    const int x0 = (tile % tiles_x) * DET_TW, y0 = (tile / tiles_x) * DET_TH;
    const int x1 = min(x0 + DET_TW, W) - 1, y1 = min(y0 + DET_TH, H) - 1;
    // Every load of this phase is issued before the first use: the counts and (speculatively) all entries of the candidate
    // lists of the cells the tile overlaps (one cell per lane, at most 32 cells of 8 pixels; <= 128 entries), the nodes and
    // the cuts of the proof.
    const int lb = 31 - __clz(g.B);                  // B is a power of two
    const int cap = det_cand_cap(g.B), cxa = x0 >> lb, cw = (x1 >> lb) - cxa + 1, cya = y0 >> lb, nc = cw * ((y1 >> lb) - cya + 1);
    const int hsel = (y0 / DET_TH) & 1;
    // e / d for e < 2^10 and d <= 48 as (e * m) >> 16, m = 2^16 / d + 1 (exact there)
    const unsigned m_cap = 65536u / (unsigned)cap + 1u, m_cw = 65536u / (unsigned)cw + 1u;
    unsigned n_l = 0;
    float M = -inf;
    if (lane < nc) {
        const int r = (int)(((unsigned)lane * m_cw) >> 16), cell = (cya + r) * g.GX + cxa + (lane - r * cw);
        n_l = cand_cnt[(g.B == 64) ? 2 * (size_t)cell + hsel : (size_t)cell];
        M = __ldg(cut + cell);
    }
    unsigned short slot[4];
#pragma unroll
    for (int sidx = 0; sidx < 4; ++sidx) {
        const int e = lane + 32 * sidx, ci = (int)(((unsigned)e * m_cap) >> 16), j = e - ci * cap;
        slot[sidx] = 0;
        if (ci < nc) {
            const int r = (int)(((unsigned)ci * m_cw) >> 16), cell = (cya + r) * g.GX + cxa + (ci - r * cw);
            slot[sidx] = cand_list[((g.B == 64) ? 2 * (size_t)cell + hsel : (size_t)cell) * cap + j];
        }
    }
    int gxa, gxb, gya, gyb;
    float t;
    det_node(x0, g, g.GX, gxa, t); det_node(x1, g, g.GX, gxb, t);
    det_node(y0, g, g.GY, gya, t); det_node(y1, g, g.GY, gyb, t);
    gxb = min(gxb + 1, g.GX - 1); gyb = min(gyb + 1, g.GY - 1);
    const int nw = gxb - gxa + 1, nn = nw * (gyb - gya + 1);
    const unsigned m_nw = 65536u / (unsigned)nw + 1u;
    float L = inf, A = 0.f;
    for (int e = lane; e < nn; e += 32) {
        const int r = (int)(((unsigned)e * m_nw) >> 16), q = (gya + r) * g.GX + gxa + (e - r * nw);
        const float n = __ldg(g.nse + q), b = __ldg(g.bkg + q);
        if (n < inf) { L = fminf(L, fmaf(g.k_sigma, n, b)); A = fmaxf(A, fmaf(g.k_sigma, n, fabsf(b))); }
    }
    unsigned off = n_l;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const unsigned o = __shfl_up_sync(0xffffffffu, off, d);
        if (lane >= d) off += o;
    }
    const unsigned cnt = __shfl_sync(0xffffffffu, off, 31);
    off -= n_l;
#pragma unroll
    for (int d = 16; d; d >>= 1) {
        L = fminf(L, __shfl_xor_sync(0xffffffffu, L, d));
        A = fmaxf(A, __shfl_xor_sync(0xffffffffu, A, d));
        M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, d));
    }
    // L = +inf: no defined noise node, nothing can be a source; M = -inf: every good pixel is a candidate
    const bool complete = cnt <= DET_CAND_CAP && !__any_sync(0xffffffffu, n_l > (unsigned)cap) &&
                          ((L == inf) || (M == -inf) || (L - 4e-6f * (A + fabsf(M)) - 1e-30f >= M));
    if (!complete) {
        if (lane == 0) fb_list[atomicAdd(fb_count, 1u)] = (unsigned)tile;
        return;
    }
    __shared__ uint4 s_rec[8][2 * DET_CAND_CAP];
    __shared__ unsigned short s_list[8][DET_CAND_CAP];
    uint4* rec = s_rec[threadIdx.x >> 5];
    unsigned short* mine = s_list[threadIdx.x >> 5];
#pragma unroll
    for (int sidx = 0; sidx < 4; ++sidx) {
        const int e = lane + 32 * sidx, ci = (int)(((unsigned)e * m_cap) >> 16), j = e - ci * cap;
        const unsigned n_c = __shfl_sync(0xffffffffu, n_l, ci & 31), off_c = __shfl_sync(0xffffffffu, off, ci & 31);
        if (ci < nc && (unsigned)j < n_c) mine[off_c + j] = slot[sidx];
    }
    __syncwarp();
    const unsigned flags = !FUSED ? det_cand_tile<0>(f, W, H, g, x0, y0, cnt, mine, rec, lane)
                           : f.pre ? det_cand_tile<2>(f, W, H, g, x0, y0, cnt, mine, rec, lane)
                                   : det_cand_tile<1>(f, W, H, g, x0, y0, cnt, mine, rec, lane);
    const int my_n = __popc(flags);
    int inc = my_n;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int o = __shfl_up_sync(0xffffffffu, inc, d);
        if (lane >= d) inc += o;
    }
    const int tile_cnt = __shfl_sync(0xffffffffu, inc, 31);
    unsigned base = 0;
    if (lane == 0) {
        base = tile_cnt ? atomicAdd(total, (unsigned)tile_cnt) : 0u;
        if (tile_cnt) atomicAdd(band_cnt + tile / tiles_x, (unsigned)tile_cnt);
        tile_info[tile] = make_uint2(base, (unsigned)tile_cnt);
    }
    base = __shfl_sync(0xffffffffu, base, 0);
    unsigned pos = base + (unsigned)(inc - my_n);
    for (unsigned it = 0; flags >> it; ++it) {
        if (!((flags >> it) & 1u)) continue;
        if (pos < capacity) {
            uint4* dst = reinterpret_cast<uint4*>(tmp + pos);
            dst[0] = rec[2 * (it * 32 + lane)];
            dst[1] = rec[2 * (it * 32 + lane) + 1];
        }
        ++pos;
    }
}

// (used by argus_subtract_tiles; detection folds this scan into det_order_kernel)
// Exclusive scan of the tile counts in tile order; *n_dev (may be NULL) and ctl[1] receive the total.  One CTA of
// 1024 threads; 16 x 1024 tiles per round: every thread loads its (coalesced) element of all 16 chunks at once, scans
// each within its warp, the 16 x 32 warp totals are scanned once by the whole CTA -- five barriers per round instead
// of four per chunk (a 61-MPix frame has 30 000 tiles: two rounds).
__global__ void __launch_bounds__(1024) det_scan_kernel(const uint2* __restrict__ tile_info, int n_tiles,
                                                        unsigned* __restrict__ offsets, unsigned* __restrict__ ctl,
                                                        long long* __restrict__ n_dev) {
    constexpr int NB = 16;                            // chunks of 1024 tiles per round
    __shared__ unsigned s_tot[1024];                  // [chunk][warp] inclusive warp totals -> exclusive prefixes (NB * 32 used)
    __shared__ unsigned s_w[32];
    __shared__ unsigned s_carry;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    if (tid == 0) s_carry = 0;
    __syncthreads();
    for (int base = 0; base < n_tiles; base += NB * 1024) {
        unsigned exc[NB];                              // exclusive prefix inside the warp
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const int i = base + b * 1024 + tid;
            exc[b] = i < n_tiles ? tile_info[i].y : 0u;
        }
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            unsigned x = exc[b];
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const unsigned o = __shfl_up_sync(0xffffffffu, x, d);
                if (lane >= d) x += o;
            }
            if (lane == 31) s_tot[b * 32 + wid] = x;
            exc[b] = x - exc[b];
        }
        __syncthreads();
        // scan the 1024 warp totals in (chunk, warp) order: thread t owns total t
        const unsigned t = tid < NB * 32 ? s_tot[tid] : 0u;
        unsigned x = t;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned o = __shfl_up_sync(0xffffffffu, x, d);
            if (lane >= d) x += o;
        }
        if (lane == 31) s_w[wid] = x;
        __syncthreads();
        if (wid == 0) {
            const unsigned v = s_w[lane];
            unsigned y = v;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const unsigned o = __shfl_up_sync(0xffffffffu, y, d);
                if (lane >= d) y += o;
            }
            s_w[lane] = y - v;
        }
        __syncthreads();
        const unsigned carry = s_carry;
        s_tot[tid] = carry + s_w[wid] + x - t;        // exclusive prefix of (chunk, warp) total `tid`
        __syncthreads();
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const int i = base + b * 1024 + tid;
            if (i < n_tiles) offsets[i] = s_tot[b * 32 + wid] + exc[b];
        }
        if (tid == 1023) s_carry = carry + s_w[31] + x;
        __syncthreads();
    }
    if (tid == 0) {
        ctl[1] = s_carry;
        if (n_dev) *n_dev = (long long)s_carry;
    }
}

// Count-only calls: the number of sources (the running total of the tile kernels) to the caller's device word.
__global__ void det_count_kernel(const unsigned* __restrict__ ctl, long long* __restrict__ n_dev) {
    if (n_dev) *n_dev = (long long)ctl[0];
}

// Catalogue order (R-D6: ascending raster index y * W + x).  The tile kernels leave every tile's records at an arbitrary
// base of tmp (in any order inside the tile) and the number of records of every tile row ("band", DET_TH image rows) in
// band_cnt.  One CTA per band: (0) start of the band in the catalogue = sum of the earlier bands' counts, start of every tile
// inside it = running sum of the tile counts (to offsets[]: no separate scan kernel); (1) band-local keys (y - y0) * W + x
// (< 2^25) and source positions of the band's records to scratch; (2) rank of every record = number of smaller keys in the
// band (keys are unique), counted against chunks of 1024 keys staged in shared memory (a 61-MPix frame has ~160 records
// per band); (3) record -> out[band start + rank].  The last band stores the total in *n_dev.
#define DET_ORD_CHUNK 1024
__global__ void __launch_bounds__(256) det_order_kernel(const uint2* __restrict__ tile_info, unsigned* __restrict__ offsets,
                                                        int n_tiles, int tiles_x, int W, const unsigned* __restrict__ band_cnt,
                                                        const ArgusSourceRec* __restrict__ tmp, uint2* __restrict__ ord,
                                                        ArgusSourceRec* __restrict__ out, unsigned capacity,
                                                        long long* __restrict__ n_dev) {
    __shared__ unsigned s_key[DET_ORD_CHUNK];
    __shared__ unsigned s_w[8], s_carry;
    const int band = blockIdx.x, t0 = band * tiles_x, t1 = min(t0 + tiles_x, n_tiles);
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    // (0) band start
    unsigned part = 0;
    for (int b = tid; b < band; b += 256) part += band_cnt[b];
    part = __reduce_add_sync(0xffffffffu, part);
    if (lane == 0) s_w[wid] = part;
    __syncthreads();
    unsigned band_off = 0;
#pragma unroll
    for (int w = 0; w < 8; ++w) band_off += s_w[w];
    const unsigned n_band = band_cnt[band], band_end = band_off + n_band;
    if (band == (int)gridDim.x - 1 && tid == 0 && n_dev) *n_dev = (long long)band_end;
    if (band_end > capacity) {
        if (band_off >= capacity) return;       // overflow: the contents of out are unspecified, nothing beyond capacity
    }
    const unsigned n_b = min(band_end, capacity) - band_off;
    if (n_b == 0) return;
    // tile starts: exclusive scan of the band's tile counts, 256 tiles per round
    if (tid == 0) s_carry = band_off;
    __syncthreads();
    for (int c0 = t0; c0 < t1; c0 += 256) {
        const int tile = c0 + tid;
        const unsigned cnt = tile < t1 ? tile_info[tile].y : 0u;
        unsigned inc = cnt;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned o = __shfl_up_sync(0xffffffffu, inc, d);
            if (lane >= d) inc += o;
        }
        if (lane == 31) s_w[wid] = inc;
        __syncthreads();
        unsigned before = s_carry;
#pragma unroll
        for (int w = 0; w < 8; ++w) before += (w < wid) ? s_w[w] : 0u;
        if (tile < t1) offsets[tile] = before + inc - cnt;
        __syncthreads();
        if (tid == 255) s_carry = before + inc;
    }
    __syncthreads();
    const int y0 = band * DET_TH;
    for (int tile = t0 + wid; tile < t1; tile += 8) {
        const uint2 info = tile_info[tile];
        const unsigned off = offsets[tile];
        for (unsigned j = lane; j < info.y; j += 32) {
            if (info.x + j >= capacity || off + j >= capacity) break;
            const int2 xy = *reinterpret_cast<const int2*>(tmp + info.x + j);
            ord[off + j] = make_uint2((unsigned)((xy.y - y0) * W + xy.x), info.x + j);
        }
    }
    __syncthreads();
    for (unsigned i0 = 0; i0 < n_b; i0 += 256) {
        const unsigned i = i0 + tid;
        const uint2 mine = i < n_b ? ord[band_off + i] : make_uint2(0u, 0u);
        unsigned rank = 0;
        for (unsigned c0 = 0; c0 < n_b; c0 += DET_ORD_CHUNK) {
            const unsigned m = min((unsigned)DET_ORD_CHUNK, n_b - c0);
            __syncthreads();
            for (unsigned e = tid; e < m; e += 256) s_key[e] = ord[band_off + c0 + e].x;
            __syncthreads();
            for (unsigned e = 0; e < m; ++e) rank += (s_key[e] < mine.x) ? 1u : 0u;
        }
        if (i < n_b && rank < n_b && mine.y < capacity) {   // (garbage entries exist only after a capacity overflow)
            const uint4* src = reinterpret_cast<const uint4*>(tmp + mine.y);
            uint4* dst = reinterpret_cast<uint4*>(out + band_off + rank);
            dst[0] = src[0];
            dst[1] = src[1];
        }
    }
}
