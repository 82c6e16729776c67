// plan_block.cuh -- A0/A1, hierarchical front end of the plan: the sky->pixel mapping is fitted ONCE per block of
// 8 x 8 tiles (256 x 256 HEALPix pixels = 65536 consecutive nested indices) from 32 exact FP64 evaluations, and
// every tile's cubic is obtained from the block's quartic by re-expansion about the tile centre -- 64 times fewer
// exact evaluations than one fit per tile.  (Measured: a total-degree-4 fit over 256 px leaves
// <= 2e-9 px, the quartic terms dropped by the re-expansion are 8^-4 of that scale.)
//
//   bscan    : every block-level child of the host-chosen coarse cells is tested with one exact evaluation of its
//              centre; the last CTA to finish compacts the survivors into the ascending block list
//   blockfit : one warp per block: 25 nodes + 7 check points -> least-squares quartic, residual check
//   tilegen  : one thread per tile: re-expansion, extent from the tile corners, classification, tile records.
//              Blocks that are not smooth (belt/cap ring, poles), not inside the search cone or badly fitted hand
//              their 64 tiles to plan_fit_kernel (one fit per tile, list mode).
// Tile index t = 64 * (position of the block) + (tile's Morton index in the block): ascending nested order.
#pragma once
#include "plan.cuh"

#define BLOCK_TILES_LOG2 3                 // block = 8 x 8 tiles
#define BLOCK_PIX 256

// ------------------------------------------------------------------------------------------- bscan
__global__ void __launch_bounds__(256) plan_bscan_kernel(DevWcs w, CoarseList cl, PlanBuffers pb, double rad_px, double block_ang) {
    __shared__ int s_last;
    __shared__ int s_part[8];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int rl = cl.ratio_log2;                                  // block-level cells per coarse cell = 4^rl
    const long long n_slots = (long long)cl.n << (2 * rl);
    const long long slot = (long long)blockIdx.x * 256 + tid;
    const int kb = w.k - ARGUS_TILE_LOG2 - BLOCK_TILES_LOG2;       // log2 of the block-level nside
    int keep = 0;
    if (slot < n_slots) {
        const int c = (int)(slot >> (2 * rl));
        const long long blk = (cl.cell[c] << (2 * rl)) | (slot & ((1ll << (2 * rl)) - 1));
        int face, bx, by;
        nest_to_xyf(blk, kb, face, bx, by);
        const double ixc = bx * 256.0 + 127.5, iyc = by * 256.0 + 127.5;
        const long long ns = 1ll << w.k;
        const long long jr = (long long)face_ring_offset(face) * ns - (long long)(ixc + iyc) - 1;
        double v[3], x, y;
        hp_vec(face, ixc, iyc, w.nside, ring_zone(jr, ns), v);
        const double cosc = vec_to_xy(w, v, x, y);
        if (cosc > 0.05 && acos(fmin(cosc, 1.0)) <= w.rho + block_ang)
            keep = (x >= -0.5 - rad_px) && (x < w.W - 0.5 + rad_px) && (y >= -0.5 - rad_px) && (y < w.H - 0.5 + rad_px);
        pb.slot_flag[slot] = (unsigned char)keep;
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = (atomicAdd(pb.ticket, 1u) == gridDim.x - 1);
    __syncthreads();
    if (!s_last) return;
    // ---- last CTA: order-preserving compaction of all slots, reset of the per-plan counters
    __threadfence();
    if (tid == 0) pb.stats->overflow = 0;
    __syncthreads();
    // 8 consecutive slots per thread and pass (flags read as one 64-bit word: slot_flag is 256-byte aligned)
    int base = 0;
    for (long long s0 = 0; s0 < n_slots; s0 += 2048) {
        const long long s = s0 + 8ll * tid;
        unsigned long long fl8 = 0ull;
        if (s < n_slots) fl8 = __ldcg(reinterpret_cast<const unsigned long long*>(pb.slot_flag + s));
        if (s + 8 > n_slots && s < n_slots) fl8 &= (1ull << (8 * (int)(n_slots - s))) - 1ull;   // tail: stale bytes beyond n_slots
        const int cnt = __popcll(fl8 & 0x0101010101010101ull);
        int inc = cnt;
        for (int o = 1; o < 32; o <<= 1) {
            const int y = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += y;
        }
        if (lane == 31) s_part[wid] = inc;
        __syncthreads();
        int woff = 0, tot = 0;
        for (int i = 0; i < 8; ++i) { if (i < wid) woff += s_part[i]; tot += s_part[i]; }
        int pos = base + woff + inc - cnt;
        for (int j = 0; j < 8; ++j)
            if ((fl8 >> (8 * j)) & 1ull) {
                if ((long long)(pos + 1) * 64 <= pb.max_tiles) {
                    const long long sj = s + j;
                    const int c = (int)(sj >> (2 * rl));
                    pb.block_id[pos] = (cl.cell[c] << (2 * rl)) | (sj & ((1ll << (2 * rl)) - 1));
                } else {
                    plan_overflow(pb, 1);
                }
                ++pos;
            }
        base += tot;
        __syncthreads();
    }
    if (tid == 0) {
        int nb = base;
        if ((long long)nb * 64 > pb.max_tiles) nb = pb.max_tiles / 64;
        *pb.n_blocks = nb;
        *pb.n_tiles = nb * 64;
        *pb.ticket = 0u;
        *pb.hard_count = 0;
        *pb.slow_count = 0;
        *pb.fb_count = 0;
        PlanStats* st = pb.stats;
        st->n_inside = st->n_border = st->n_exact = st->n_empty = 0;
    }
}

// ---------------------------------------------------------------------------------------- blockfit
__device__ __forceinline__ constexpr int q_idx(int i, int j) { return (i + j) * (i + j + 1) / 2 + j; }   // U^i V^j
__device__ __forceinline__ constexpr int binom(int n, int k) {
    return k == 0 ? 1 : (k == 1 ? n : (k == 2 ? n * (n - 1) / 2 : (k == 3 ? n * (n - 1) * (n - 2) / 6 : 1)));
}

// Cubic of a tile from the block's quartic p[15] (basis U^i V^j, U, V in [-1, 1] over the block): U = Uc + S/8,
// V = Vc + T/8; terms of local degree 4 are dropped (8^-4 of the quartic's size).
__device__ inline void reexpand_cubic(const double* __restrict__ p, double Uc, double Vc, double* __restrict__ c) {
    double Up[5], Vp[5];
    Up[0] = Vp[0] = 1.0;
#pragma unroll
    for (int i = 1; i < 5; ++i) { Up[i] = Up[i - 1] * Uc; Vp[i] = Vp[i - 1] * Vc; }
#pragma unroll
    for (int m = 0; m <= 3; ++m)
#pragma unroll
        for (int n = 0; n + m <= 3; ++n) {
            double acc = 0.0;
#pragma unroll
            for (int i = m; i <= 4; ++i)
#pragma unroll
                for (int j = n; i + j <= 4; ++j)
                    acc = fma(p[q_idx(i, j)] * (double)(binom(i, m) * binom(j, n)), Up[i - m] * Vp[j - n], acc);
            double sc = 1.0;
#pragma unroll
            for (int e = 0; e < m + n; ++e) sc *= 0.125;
            c[q_idx(m, n)] = acc * sc;
        }
}

#define BFIT_WARPS 4
__global__ void __launch_bounds__(32 * BFIT_WARPS) plan_blockfit_kernel(DevWcs w, PlanBuffers pb) {
    __shared__ double s_pinv[375];
    __shared__ double s_bc[BFIT_WARPS][30];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    for (int i = tid; i < 375; i += blockDim.x) s_pinv[i] = pb.pinv4[i];
    __syncthreads();
    const int n_blocks = *pb.n_blocks;
    const long long ns = 1ll << w.k;
    const int kb = w.k - ARGUS_TILE_LOG2 - BLOCK_TILES_LOG2;
    double S, T;   // lanes 0..24 the 5x5 fit grid, lanes 25..31 extra check points
    if (lane < 25) {
        S = -1.0 + 0.5 * (lane % 5);
        T = -1.0 + 0.5 * (lane / 5);
    } else {
        const double cs[7] = {0.77, -0.77, 0.33, -0.33, 0.9, -0.2, 0.61};
        const double ct[7] = {0.33, 0.61, -0.77, -0.9, 0.9, 0.15, -0.41};
        S = cs[lane - 25];
        T = ct[lane - 25];
    }
    for (int b = blockIdx.x * BFIT_WARPS + wid; b < n_blocks; b += gridDim.x * BFIT_WARPS) {
        const long long blk = pb.block_id[b];
        int face, bx, by;
        nest_to_xyf(blk, kb, face, bx, by);
        const int ix0 = bx * BLOCK_PIX, iy0 = by * BLOCK_PIX;
        const long long jr_max = (long long)face_ring_offset(face) * ns - ix0 - iy0 - 1, jr_min = jr_max - 2 * (BLOCK_PIX - 1);
        const int z0 = ring_zone(jr_min, ns), z1 = ring_zone(jr_max, ns);
        bool ok = (z0 == z1);
        if (ok) {
            double v[3], x, y;
            hp_vec(face, ix0 + 127.5 + 128.0 * S, iy0 + 127.5 + 128.0 * T, w.nside, z0, v);
            const double cosc = vec_to_xy(w, v, x, y);
            const double amax = warp_max(fmax(fabs(x), fabs(y)));
            const double cmin = warp_min(cosc);
            const double xc = __shfl_sync(0xffffffffu, x, 12), yc = __shfl_sync(0xffffffffu, y, 12);
            // least squares: lanes 0..14 -> x coefficients, lanes 15..29 -> y coefficients
            double acc = 0.0;
            const int row = lane < 15 ? lane : lane - 15;
            for (int n = 0; n < 25; ++n) {
                const double xn = __shfl_sync(0xffffffffu, x, n) - xc, yn = __shfl_sync(0xffffffffu, y, n) - yc;
                if (lane < 30) acc = fma(s_pinv[row * 25 + n], lane < 15 ? xn : yn, acc);
            }
            if (lane == 0) acc += xc;
            if (lane == 15) acc += yc;
            if (lane < 30) s_bc[wid][lane] = acc;
            __syncwarp();
            double fxv = 0.0, fyv = 0.0;
            {
                double Sp[5], Tp[5];
                Sp[0] = Tp[0] = 1.0;
#pragma unroll
                for (int i = 1; i < 5; ++i) { Sp[i] = Sp[i - 1] * S; Tp[i] = Tp[i - 1] * T; }
#pragma unroll
                for (int i = 0; i <= 4; ++i)
#pragma unroll
                    for (int j = 0; i + j <= 4; ++j) {
                        const double mono = Sp[i] * Tp[j];
                        fxv = fma(s_bc[wid][q_idx(i, j)], mono, fxv);
                        fyv = fma(s_bc[wid][15 + q_idx(i, j)], mono, fyv);
                    }
            }
            const double res = warp_max(fmax(fabs(fxv - x), fabs(fyv - y)));
            const bool cone_in = acos(fmin(cmin, 1.0)) + 0.1 * w.tile_ang <= w.rho;   // nodes include the block corners
            ok = (amax < 1e8) && (cmin > 0.05) && (res <= PLAN_FIT_TOL) && cone_in;   // NaN compares false
        }
        // hand over to plan_tilegen_kernel: 30 coefficients (x then y) + status word (zone, or -1 = no block fit)
        if (lane < 30) pb.bcoef[(size_t)b * 32 + lane] = ok ? s_bc[wid][lane] : 0.0;
        if (lane == 30) pb.bcoef[(size_t)b * 32 + 30] = ok ? (double)z0 : -1.0;
        __syncwarp();
    }
}

// ----------------------------------------------------------------------------------------- tilegen
// One thread per tile: re-expansion of the block quartic about the tile centre, extent from the tile corners,
// classification, tile records.  Tiles of blocks without a fit go to the per-tile fit list.
__global__ void __launch_bounds__(128, 4) plan_tilegen_kernel(DevWcs w, PlanBuffers pb, int lite) {
    __shared__ double s_bc[2][32];
    const int tid = threadIdx.x;
    const int n_blocks = *pb.n_blocks;
    for (int b0 = blockIdx.x * 2; b0 < n_blocks; b0 += gridDim.x * 2) {
        __syncthreads();
        if (tid < 64) {
            const int b = b0 + (tid >> 5);
            s_bc[tid >> 5][tid & 31] = (b < n_blocks) ? pb.bcoef[(size_t)b * 32 + (tid & 31)] : -1.0;
        }
        __syncthreads();
        const int half = tid >> 6, j = tid & 63, b = b0 + half;
        if (b >= n_blocks) continue;
        const long long blk = pb.block_id[b];
        const int t = b * 64 + j;
        const long long tile = (blk << 6) | j;
        const double* bc = s_bc[half];
        if (bc[30] < 0.0) {
            pb.tile_id[t] = tile;
            const int fb = atomicAdd(pb.fb_count, 1);      // fb < 64 n_blocks <= max_tiles
            pb.fb_list[fb] = t;
            continue;
        }
        const int ta = (int)compact_even_bits((unsigned)j), tb = (int)compact_even_bits((unsigned)j >> 1);
        const double Uc = ((double)ta - 3.5) * 0.25, Vc = ((double)tb - 3.5) * 0.25;
        double c[20];
        reexpand_cubic(bc, Uc, Vc, c);
        reexpand_cubic(bc + 15, Uc, Vc, c + 10);
        // extent of the source positions: the four tile corners (S, T = +-1) plus the size of the nonlinear part
        double xmin = 1e300, xmax = -1e300, ymin = 1e300, ymax = -1e300;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const double s = (q & 1) ? 1.0 : -1.0, tt = (q >> 1) ? 1.0 : -1.0;
            double m[10];
            cubic_basis(s, tt, m);
            double xv = 0.0, yv = 0.0;
#pragma unroll
            for (int i = 0; i < 10; ++i) { xv = fma(c[i], m[i], xv); yv = fma(c[10 + i], m[i], yv); }
            xmin = fmin(xmin, xv); xmax = fmax(xmax, xv); ymin = fmin(ymin, yv); ymax = fmax(ymax, yv);
        }
        double nl = 0.0;
#pragma unroll
        for (int i = 3; i < 10; ++i) nl += fmax(fabs(c[i]), fabs(c[10 + i]));
        const double mg = PLAN_NODE_MARGIN + nl;
        const bool all_out = (xmax + mg < -0.5) || (xmin - mg >= w.W - 0.5) || (ymax + mg < -0.5) || (ymin - mg >= w.H - 0.5);
        const bool all_in = (xmin - mg >= -0.5) && (xmax + mg < w.W - 0.5) && (ymin - mg >= -0.5) && (ymax + mg < w.H - 0.5);
        const int cls = all_out ? TC_EMPTY : (all_in ? TC_INSIDE : TC_BORDER);
        emit_tile(pb, t, tile, (int)bc[30], cls, c, xmin, xmax, ymin, ymax, mg, lite != 0);
    }
}
