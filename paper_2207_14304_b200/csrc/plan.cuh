// plan.cuh -- A0/A1: the per-frame resampling plan, built entirely on the device (no host sync).
//
//   scan    : every tile-level child of the host-chosen coarse cells is tested with one exact FP64
//             evaluation of its centre (conservative radius) -> flag + per-block count
//   compact : order-preserving compaction -> ascending list of candidate tiles
//   fit     : one warp per tile: 25 exact nodes -> least-squares cubic in local coordinates, residual
//             check against 7 extra exact points, classification (inside / border / exact / empty)
//   members : border / exact tiles: per-pixel membership mask (exact FP64 decision inside a guard band),
//             count and source bounding box
//   offsets : exclusive scan of the per-tile counts -> output positions, statistics
//
// The footprint (A1) is represented as this range plan; argus_healpix_footprint expands it
// into the explicit ascending int64 list on request.
#pragma once
#include "common.cuh"

#define PLAN_GUARD_PX 2e-5f      // |distance to the domain border| below which membership is decided in FP64
#define PLAN_FIT_TOL 3e-8        // max residual (px) of the cubic fit at the 32 exact points
#define PLAN_NODE_MARGIN 0.25    // px margin on node extents for the inside / empty classification

struct PlanBuffers {
    unsigned char* slot_flag;   // [max_slots]
    int* block_count;           // [max_slots/256]
    long long* tile_id;         // [max_tiles]
    TileRec* rec;               // [max_tiles]
    int* tile_count;            // [max_tiles]
    int* tile_offset;           // [max_tiles] exclusive prefix of tile_count inside its block of 1024 tiles
    unsigned char* tile_cls;    // [max_tiles] compact copy of TileRec.cls
    int* block_sum;             // [max_tiles/1024 + 1]
    long long* block_base;      // [max_tiles/1024 + 1] exclusive prefix of block_sum
    int* n_tiles;               // device scalar
    int* hard_count;            // device scalar
    int* hard_list;             // [max_hard] tile positions
    unsigned* masks;            // [max_hard][32]
    PlanStats* stats;           // device
    double* pinv;               // [10][25] least-squares pseudo-inverse of the node design matrix
    double* dcoef;              // [max_tiles][20] unsplit FP64 polynomial coefficients (x then y)
    FastRec* frec;              // [max_tiles] records of the TMA-staged bilinear kernel
    int* slow_count;            // device scalar
    int* slow_plan;             // device scalar: slow_count as the plan left it; the Lanczos-3 fast kernel appends behind
                                // it at run time and the general kernel restores it when it is done (a cached plan is reused)
    int* slow_list;             // [max_tiles] tiles the fast kernel leaves to the general kernel
    long long* cslot;           // [max_tiles] coadd slot of each tile's first pixel for the layout of the current call (-1 = absent)
    int* latch;                 // context-wide: every overflow bit is also ORed in here; cleared only when read
    long long* block_id;        // [max_tiles/64] candidate blocks (8x8 tiles), ascending nested ids at block level
    int* n_blocks;              // device scalar
    int* fb_count;              // device scalar
    int* fb_list;               // [max_tiles] tiles of blocks that need one fit per tile
    unsigned* ticket;           // device scalar: CTA arrival counter of plan_bscan_kernel
    double* pinv4;              // [15][25] pseudo-inverse of the quartic design matrix on the 5x5 node grid
    double* bcoef;              // [max_tiles/64][32] block quartics (15 x, 15 y), [30] = zone or -1 (no block fit)
    int max_slots, max_tiles, max_hard;
    int fast_tl, fast_tr, fast_cap;   // tap apron and stage capacity (pixels) of the fast kernel this plan is for
    int unit_mode;                    // the image-aligned unit kernel runs the frame: no per-tile box limits (resample_unit.cuh)
};

// Overflow bits (PlanStats.overflow) live in the plan slot and are zeroed by the next plan into it; the context-wide
// latch keeps them until argus_plan_info / argus_healpix_footprint reads them.
__device__ inline void plan_overflow(const PlanBuffers& pb, int bits) {
    atomicOr(&pb.stats->overflow, bits);
    atomicOr(pb.latch, bits);
}

// --------------------------------------------------------------------------------------------- scan
__global__ void __launch_bounds__(256) plan_scan_kernel(DevWcs w, CoarseList cl, PlanBuffers pb, double rad_px) {
    long long slot = (long long)blockIdx.x * 256 + threadIdx.x;
    long long n_slots = (long long)cl.n << (2 * cl.ratio_log2);
    int keep = 0;
    if (slot < n_slots) {
        int c = (int)(slot >> (2 * cl.ratio_log2));
        long long tile = (cl.cell[c] << (2 * cl.ratio_log2)) | (slot & ((1ll << (2 * cl.ratio_log2)) - 1));
        int face, tx, ty;
        nest_to_xyf(tile, w.k - ARGUS_TILE_LOG2, face, tx, ty);
        double ixc = tx * 32.0 + 15.5, iyc = ty * 32.0 + 15.5;
        long long ns = 1ll << w.k;
        long long jr = (long long)face_ring_offset(face) * ns - (long long)(ixc + iyc) - 1;
        double v[3], x, y;
        hp_vec(face, ixc, iyc, w.nside, ring_zone(jr, ns), v);
        double cosc = vec_to_xy(w, v, x, y);
        if (cosc > 0.05 && acos(fmin(cosc, 1.0)) <= w.rho + w.tile_ang) {
            keep = (x >= -0.5 - rad_px) && (x < w.W - 0.5 + rad_px) && (y >= -0.5 - rad_px) && (y < w.H - 0.5 + rad_px);
        }
        pb.slot_flag[slot] = (unsigned char)keep;
    }
    int cnt = __syncthreads_count(keep);
    if (threadIdx.x == 0) pb.block_count[blockIdx.x] = cnt;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        *pb.hard_count = 0;
        *pb.slow_count = 0;
        PlanStats* st = pb.stats;
        st->overflow = 0;
        st->n_inside = st->n_border = st->n_exact = st->n_empty = 0;
    }
}

// ------------------------------------------------------------------------------------------ compact
__global__ void __launch_bounds__(256) plan_compact_kernel(CoarseList cl, PlanBuffers pb) {
    __shared__ int s_part[8];
    __shared__ int s_base;
    int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    // prefix of the block counts before this block
    int acc = 0;
    for (int b = tid; b < (int)blockIdx.x; b += 256) acc += pb.block_count[b];
    for (int o = 16; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) s_part[wid] = acc;
    __syncthreads();
    if (tid == 0) {
        int t = 0;
        for (int i = 0; i < 8; ++i) t += s_part[i];
        s_base = t;
    }
    __syncthreads();
    int base = s_base;
    __syncthreads();
    long long slot = (long long)blockIdx.x * 256 + tid;
    long long n_slots = (long long)cl.n << (2 * cl.ratio_log2);
    int keep = (slot < n_slots) ? pb.slot_flag[slot] : 0;
    unsigned bal = __ballot_sync(0xffffffffu, keep);
    if (lane == 0) s_part[wid] = __popc(bal);
    __syncthreads();
    int woff = 0;
    for (int i = 0; i < wid; ++i) woff += s_part[i];
    int pos = base + woff + __popc(bal & ((1u << lane) - 1u));
    if (keep) {
        if (pos < pb.max_tiles) {
            int c = (int)(slot >> (2 * cl.ratio_log2));
            pb.tile_id[pos] = (cl.cell[c] << (2 * cl.ratio_log2)) | (slot & ((1ll << (2 * cl.ratio_log2)) - 1));
        } else {
            plan_overflow(pb, 1);
        }
    }
    if (blockIdx.x == gridDim.x - 1 && tid == 0) {
        int total = base;
        for (int i = 0; i < 8; ++i) total += s_part[i];
        *pb.n_tiles = total < pb.max_tiles ? total : pb.max_tiles;
    }
}

// ---------------------------------------------------------------------------------------------- fit
__device__ inline double warp_min(double v) {
    for (int o = 16; o; o >>= 1) v = fmin(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ inline double warp_max(double v) {
    for (int o = 16; o; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

// monomials of the total-degree-3 basis at (S, T)
__device__ inline void cubic_basis(double S, double T, double m[10]) {
    m[0] = 1.0; m[1] = S; m[2] = T; m[3] = S * S; m[4] = S * T; m[5] = T * T;
    m[6] = S * S * S; m[7] = S * S * T; m[8] = S * T * T; m[9] = T * T * T;
}

// Staged-box geometry of the fast kernel for cells [bx0, bx1] x [by0, by1] plus the interpolation kernel's taps
// (tl to the left / above, tr to the right / below: 0, 1 bilinear; 2, 3 Lanczos-3).  The TMA box must start on a
// 16-byte boundary of every array (8 pixels of the uint16 frame), so the origin is aligned down to 8; widths come in
// steps of 8 px (40..72), heights are 48, 56, 64 or 72 rows (polar-cap tiles are taller than wide) (a TMA copy costs ~100 cycles per operation whatever its
// size, so each array is fetched with ONE box).  Returns false when the box does not fit the kernel's stage.
__device__ __host__ inline int fast_cal_pitch(int boxw) { return (boxw & 15) == 8 ? boxw : boxw + 8; }   // = 8 or 24 mod 32
__device__ inline bool fast_box(const PlanBuffers& pb, int bx0, int bx1, int by0, int by1, int X0, int Y0, FastRec& f) {
    const int tl = pb.fast_tl, tr = pb.fast_tr;
    int gx0 = (bx0 - tl) & ~7, gy0 = by0 - tl;
    int bw = bx1 + tr + 1 - gx0, bh = by1 + tr + 1 - gy0;
    if (bw < 1 || bh < 1 || bw > 72 || bh > 72) return false;
    int wclass = bw <= 40 ? 0 : (bw - 40 + 7) >> 3;
    int boxw = 40 + 8 * wclass, pitch = fast_cal_pitch(boxw);
    int hclass = bh <= 48 ? 0 : (bh - 48 + 7) >> 3;      // 48, 56, 64 or 72 rows
    if ((48 + 8 * hclass) * boxw > pb.fast_cap || bh * pitch > pb.fast_cap + pb.fast_cap / 8) return false;
    if (bx0 < X0 || by0 < Y0 || bx1 + 4 - X0 > 110 || by1 + 4 - Y0 > 110) return false;
    f.gx0 = gx0; f.gy0 = gy0; f.wclass = wclass | (hclass << 4); f.bh = bh;
    f.kofs = (Y0 - gy0) * pitch + (X0 - gx0);
    return true;
}

__device__ inline void slow_push(const PlanBuffers& pb, int t) {
    int s = atomicAdd(pb.slow_count, 1);
    if (s < pb.max_tiles) pb.slow_list[s] = t;
    else plan_overflow(pb, 2);
}

// Everything a kernel needs to know about one tile, written by ONE thread from the tile's cubic (c[0..9] x,
// c[10..19] y, in S, T = local offsets / 16 px) and the extent of its source positions.  cls on entry:
// TC_INSIDE / TC_BORDER / TC_EXACT / TC_EMPTY.
// lite: TileRec and the FP64 coefficients (used by the general kernel only) are written just for the tiles that
// kernel will visit when the fast kernel runs the frame (border / exact / oversized tiles).
__device__ inline void emit_tile(const PlanBuffers& pb, int t, long long tile, int zone, int cls, const double* c,
                                 double xmin, double xmax, double ymin, double ymax, double mg, bool lite) {
    TileRec r;
    r.tile = tile; r.reserved = 0; r.count = 0; r.mask_slot = -1;
    r.zone = zone;
    r.bx0 = r.bx1 = r.by0 = r.by1 = 0; r.X0 = r.Y0 = 0; r.ax = r.bx = r.ay = r.by = 0;
    r.pad[0] = r.pad[1] = 0;
    for (int i = 0; i < 10; ++i) { r.cx[i] = 0.f; r.cy[i] = 0.f; }
    if (cls == TC_INSIDE || cls == TC_BORDER) {
        // split: x = X0 + (a*s + b*t) 2^-12 + lo(S,T); s = 32 S, so c1 S = (c1/32) s
#pragma unroll
        for (int axis = 0; axis < 2; ++axis) {
            const double* ca = c + 10 * axis;
            double base = floor(ca[0]);
            int a = (int)rint(ca[1] * (4096.0 / 32.0)), b = (int)rint(ca[2] * (4096.0 / 32.0));
            float* out = axis ? r.cy : r.cx;
            out[0] = (float)(ca[0] - base);
            out[1] = (float)(ca[1] - a * (32.0 / 4096.0));
            out[2] = (float)(ca[2] - b * (32.0 / 4096.0));
#pragma unroll
            for (int i = 3; i < 10; ++i) out[i] = (float)ca[i];
            if (axis) { r.Y0 = (int)base; r.ay = a; r.by = b; } else { r.X0 = (int)base; r.ax = a; r.bx = b; }
        }
        r.bx0 = (int)floor(xmin - mg); r.bx1 = (int)floor(xmax + mg);
        r.by0 = (int)floor(ymin - mg); r.by1 = (int)floor(ymax + mg);
        if (cls == TC_INSIDE) r.count = ARGUS_TILE_PIX;
    }
    if (cls == TC_BORDER || cls == TC_EXACT) {
        int slot = atomicAdd(pb.hard_count, 1);
        if (slot < pb.max_hard) {
            pb.hard_list[slot] = t;
            r.mask_slot = slot;
        } else {
            plan_overflow(pb, 2);
            cls = TC_EMPTY;
        }
    }
    r.cls = cls;
    bool fast_inside = false;
    pb.tile_id[t] = tile;
    pb.tile_count[t] = r.count;
    pb.tile_cls[t] = (unsigned char)cls;
    // record of the fast (TMA-staged bilinear) kernel
    FastRec f;
    memset(&f, 0, sizeof(f));
    if (cls == TC_INSIDE || cls == TC_BORDER) {
        bool poly_ok = true;
#pragma unroll
        for (int axis = 0; axis < 2; ++axis) {
            const double* ca = c + 10 * axis;
            int base = (axis ? r.by0 : r.bx0) - 8;
            double c0l = ca[0] - (double)base;
            int c0f = (int)rint(c0l * 16777216.0);
            int af = (int)rint(ca[1] * 524288.0), bf = (int)rint(ca[2] * 524288.0);   // c/32 * 2^24
            float* pp = axis ? f.py : f.px;
            pp[0] = (float)(12582912.0 + (c0l * 16777216.0 - (double)c0f));
            pp[1] = (float)((ca[1] * 524288.0 - (double)af) * 32.0);
            pp[2] = (float)((ca[2] * 524288.0 - (double)bf) * 32.0);
            double mag = fabs((double)pp[1]) + fabs((double)pp[2]);
#pragma unroll
            for (int i = 3; i < 10; ++i) { pp[i] = (float)(ca[i] * 16777216.0); mag += fabs((double)pp[i]); }
            if (!(mag < 0.9 * 4194304.0) || !(fabs(c0l) < 100.0)) poly_ok = false;   // rounding-constant range, 32-bit range
            if (axis) { f.Y0 = base; f.c0y = c0f - FAST_MAGIC_I; f.ay = af; f.by = bf; }
            else { f.X0 = base; f.c0x = c0f - FAST_MAGIC_I; f.ax = af; f.bx = bf; }
        }
        f.mask_slot = r.mask_slot;
        f.poly_ok = poly_ok ? 1 : 0;
        if (cls == TC_INSIDE) {
            if (poly_ok && (pb.unit_mode || fast_box(pb, r.bx0, r.bx1, r.by0, r.by1, f.X0, f.Y0, f))) { f.cls = TC_INSIDE; fast_inside = true; }
            else slow_push(pb, t);
        }   // TC_BORDER: plan_members_kernel finalises the box and decides
        if (!(lite && fast_inside)) {
            double* dc = pb.dcoef + (size_t)t * 20;
#pragma unroll
            for (int i = 0; i < 20; ++i) dc[i] = c[i];
        }
    } else if (cls == TC_EXACT) {
        slow_push(pb, t);
    }
    if (lite && cls == TC_EMPTY) {
        pb.frec[t].cls = 0;                 // the fast kernel's producer only reads the class of an empty tile
    } else {
        pb.frec[t] = f;
        if (!(lite && fast_inside)) pb.rec[t] = r;
    }
}

#define FIT_WARPS 4
__global__ void __launch_bounds__(32 * FIT_WARPS) plan_fit_kernel(DevWcs w, PlanBuffers pb, int use_list, int lite) {
    __shared__ double s_pinv[250];
    __shared__ double s_coef[FIT_WARPS][20];
    int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    // use_list: only the tiles plan_blockfit_kernel could not derive from a block fit (usually none)
    const int n_items = use_list ? *pb.fb_count : *pb.n_tiles;
    if ((int)blockIdx.x * FIT_WARPS >= n_items) return;
    for (int i = tid; i < 250; i += blockDim.x) s_pinv[i] = pb.pinv[i];
    __syncthreads();
    long long ns = 1ll << w.k;
    // node coordinates: lanes 0..24 the 5x5 fit grid, lanes 25..31 extra check points
    double S, T;
    if (lane < 25) {
        S = -1.0 + 0.5 * (lane % 5);
        T = -1.0 + 0.5 * (lane / 5);
    } else {
        const double cs[7] = {0.77, -0.77, 0.33, -0.33, 0.9, -0.2, 0.61};
        const double ct[7] = {0.33, 0.61, -0.77, -0.9, 0.9, 0.15, -0.41};
        S = cs[lane - 25];
        T = ct[lane - 25];
    }
    for (int it = blockIdx.x * FIT_WARPS + wid; it < n_items; it += gridDim.x * FIT_WARPS) {
        const int t = use_list ? pb.fb_list[it] : it;
        long long tile = pb.tile_id[t];
        int face, tx, ty;
        nest_to_xyf(tile, w.k - ARGUS_TILE_LOG2, face, tx, ty);
        int ix0 = tx * 32, iy0 = ty * 32;
        long long jr_max = (long long)face_ring_offset(face) * ns - ix0 - iy0 - 1, jr_min = jr_max - 62;
        int z0 = ring_zone(jr_min, ns), z1 = ring_zone(jr_max, ns);
        double xmin = 0, xmax = 0, ymin = 0, ymax = 0;
        int cls = TC_EXACT;
        if (z0 == z1) {
            double v[3], x, y;
            hp_vec(face, ix0 + 15.5 + 16.0 * S, iy0 + 15.5 + 16.0 * T, w.nside, z0, v);
            double cosc = vec_to_xy(w, v, x, y);
            bool node = lane < 25;
            xmin = warp_min(node ? x : 1e300); xmax = warp_max(node ? x : -1e300);
            ymin = warp_min(node ? y : 1e300); ymax = warp_max(node ? y : -1e300);
            double cmin = warp_min(cosc), cmax = warp_max(cosc);
            double xc = __shfl_sync(0xffffffffu, x, 12), yc = __shfl_sync(0xffffffffu, y, 12);
            // least squares: lanes 0..9 -> x coefficients, lanes 10..19 -> y coefficients
            double acc = 0.0;
            int row = lane < 10 ? lane : lane - 10;
            for (int n = 0; n < 25; ++n) {
                double xn = __shfl_sync(0xffffffffu, x, n) - xc, yn = __shfl_sync(0xffffffffu, y, n) - yc;
                if (lane < 20) acc = fma(s_pinv[row * 25 + n], lane < 10 ? xn : yn, acc);
            }
            if (lane == 0) acc += xc;
            if (lane == 10) acc += yc;
            if (lane < 20) s_coef[wid][lane] = acc;
            __syncwarp();
            double m[10];
            cubic_basis(S, T, m);
            double fxv = 0.0, fyv = 0.0;
            for (int i = 0; i < 10; ++i) {
                fxv = fma(s_coef[wid][i], m[i], fxv);
                fyv = fma(s_coef[wid][10 + i], m[i], fyv);
            }
            double res = warp_max(fmax(fabs(fxv - x), fabs(fyv - y)));
            bool finite_ok = (xmin > -1e8) && (xmax < 1e8) && (ymin > -1e8) && (ymax < 1e8) && (cmin > 0.05);
            bool fit_ok = finite_ok && (res <= PLAN_FIT_TOL);   // NaN compares false
            double mg = PLAN_NODE_MARGIN;
            // angular distance from CRVAL is convex over the (near-planar) tile: its maximum sits on a corner
            // node; only the drop decision needs the full conservative tile radius
            bool cone_in = acos(fmin(cmin, 1.0)) + 0.1 * w.tile_ang <= w.rho;
            bool cone_out = acos(fmin(cmax, 1.0)) - w.tile_ang > w.rho;
            if (fit_ok && !cone_out) {
                bool all_out = (xmax + mg < -0.5) || (xmin - mg >= w.W - 0.5) || (ymax + mg < -0.5) || (ymin - mg >= w.H - 0.5);
                bool all_in = (xmin - mg >= -0.5) && (xmax + mg < w.W - 0.5) && (ymin - mg >= -0.5) && (ymax + mg < w.H - 0.5);
                if (all_out) cls = TC_EMPTY;
                else if (cone_in) cls = all_in ? TC_INSIDE : TC_BORDER;
                // cone-straddling tiles stay TC_EXACT
            } else if (finite_ok && cone_out) {
                cls = TC_EMPTY;
            }
        }
        if (lane == 0) emit_tile(pb, t, tile, (z0 == z1) ? z0 : -1, cls, s_coef[wid], xmin, xmax, ymin, ymax, PLAN_NODE_MARGIN, lite != 0);
        __syncwarp();
    }
}

// ------------------------------------------------------------------------------------------ members
// Thread -> 2x2 block of pixels = 4 consecutive Morton (nested) indices 4*tid .. 4*tid+3.
__device__ inline void thread_block_origin(int tid, int& u0, int& v0) {
    u0 = 2 * (int)compact_even_bits((unsigned)tid);
    v0 = 2 * (int)compact_even_bits((unsigned)tid >> 1);
}

// Membership of pixel (u, v) of a TC_BORDER tile from the tile polynomial; the decision is re-taken in
// FP64 with the exact mapping whenever the FP32 position is within PLAN_GUARD_PX of a border line.
__device__ inline bool border_member(const DevWcs& w, const PolyAxis& px, const PolyAxis& py, int face, int ix0,
                                     int iy0, int u, int v, int& ci, int& cj) {
    float fx, fy;
    poly_axis_eval(px, 2 * u - 31, 2 * v - 31, ci, fx);
    poly_axis_eval(py, 2 * u - 31, 2 * v - 31, cj, fy);
    bool near = ((ci == -1 || ci == w.W - 1) && fabsf(fx - 0.5f) < PLAN_GUARD_PX) ||
                ((cj == -1 || cj == w.H - 1) && fabsf(fy - 0.5f) < PLAN_GUARD_PX);
    if (near) {
        double x, y;
        double cosc = pixel_to_xy(w, face, ix0 + u, iy0 + v, x, y);
        return in_domain(w, cosc, x, y);
    }
    bool inx = (ci >= 0 || (ci == -1 && fx >= 0.5f)) && (ci < w.W - 1 || (ci == w.W - 1 && fx < 0.5f));
    bool iny = (cj >= 0 || (cj == -1 && fy >= 0.5f)) && (cj < w.H - 1 || (cj == w.H - 1 && fy < 0.5f));
    return inx && iny;
}

__global__ void __launch_bounds__(256, 4) plan_members_kernel(DevWcs w, PlanBuffers pb) {
    __shared__ unsigned s_mask[32];
    __shared__ int s_wext[8][5];     // per warp: xmin, xmax, ymin, ymax, count
    __shared__ TileRec s_rec;
    int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    int n_hard = *pb.hard_count;
    if (n_hard > pb.max_hard) n_hard = pb.max_hard;
    int u0, v0;
    thread_block_origin(tid, u0, v0);
    for (int h = blockIdx.x; h < n_hard; h += gridDim.x) {
        int t = pb.hard_list[h];
        __syncthreads();
        if (tid < (int)(sizeof(TileRec) / 16)) reinterpret_cast<int4*>(&s_rec)[tid] = __ldg(reinterpret_cast<const int4*>(pb.rec + t) + tid);
        __syncthreads();
        const TileRec& r = s_rec;
        int face, tx, ty;
        nest_to_xyf(r.tile, w.k - ARGUS_TILE_LOG2, face, tx, ty);
        int ix0 = tx * 32, iy0 = ty * 32;
        int cls = r.cls;
        PolyAxis px, py;
        if (cls == TC_BORDER) { poly_axis_load(r, 0, px); poly_axis_load(r, 1, py); }
        unsigned nib = 0;
        int xmin = 0x7fffffff, xmax = -0x7fffffff, ymin = 0x7fffffff, ymax = -0x7fffffff;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            int u = u0 + (q & 1), v = v0 + (q >> 1);
            int ci, cj;
            bool in;
            if (cls == TC_BORDER) {
                in = border_member(w, px, py, face, ix0, iy0, u, v, ci, cj);
            } else {
                double x, y;
                double cosc = pixel_to_xy(w, face, ix0 + u, iy0 + v, x, y);
                in = in_domain(w, cosc, x, y);
                ci = in ? (int)floor(x) : 0;
                cj = in ? (int)floor(y) : 0;
            }
            if (in) {
                nib |= 1u << q;
                xmin = min(xmin, ci); xmax = max(xmax, ci); ymin = min(ymin, cj); ymax = max(ymax, cj);
            }
        }
        // warp-level reductions (no shared-memory atomics): 8 threads make one mask word
        unsigned word = nib << (4 * (tid & 7));
        word |= __shfl_xor_sync(0xffffffffu, word, 1);
        word |= __shfl_xor_sync(0xffffffffu, word, 2);
        word |= __shfl_xor_sync(0xffffffffu, word, 4);
        if ((tid & 7) == 0) s_mask[tid >> 3] = word;
        xmin = __reduce_min_sync(0xffffffffu, xmin); xmax = __reduce_max_sync(0xffffffffu, xmax);
        ymin = __reduce_min_sync(0xffffffffu, ymin); ymax = __reduce_max_sync(0xffffffffu, ymax);
        int cnt = __reduce_add_sync(0xffffffffu, __popc(nib));
        if (lane == 0) { s_wext[wid][0] = xmin; s_wext[wid][1] = xmax; s_wext[wid][2] = ymin; s_wext[wid][3] = ymax; s_wext[wid][4] = cnt; }
        __syncthreads();
        if (tid < 32) pb.masks[(size_t)h * 32 + tid] = s_mask[tid];
        if (tid == 0) {
            int e0 = 0x7fffffff, e1 = -0x7fffffff, e2 = 0x7fffffff, e3 = -0x7fffffff, c = 0;
            for (int i = 0; i < 8; ++i) {
                e0 = min(e0, s_wext[i][0]); e1 = max(e1, s_wext[i][1]); e2 = min(e2, s_wext[i][2]); e3 = max(e3, s_wext[i][3]);
                c += s_wext[i][4];
            }
            TileRec* wr = &pb.rec[t];
            wr->count = c;
            pb.tile_count[t] = c;
            if (c == 0) {
                wr->cls = TC_EMPTY;
                pb.tile_cls[t] = TC_EMPTY;
            } else {
                wr->bx0 = e0; wr->bx1 = e1; wr->by0 = e2; wr->by1 = e3;
                if (cls == TC_BORDER) {
                    FastRec* fr = &pb.frec[t];
                    FastRec f = *fr;
                    if (f.poly_ok && (pb.unit_mode || fast_box(pb, e0, e1, e2, e3, f.X0, f.Y0, f))) {
                        f.cls = TC_BORDER;
                        *fr = f;
                    } else {
                        slow_push(pb, t);
                    }
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------ offsets
// Exclusive scan of the per-tile counts in one launch: block-local scan (1024 tiles per CTA, coalesced reads of
// the compact count / class arrays); the last CTA to finish scans the per-CTA sums.
// Output position of tile t = block_base[t >> 10] + tile_offset[t].
__device__ inline void offsets_final_body(const PlanBuffers& pb, long long out_capacity, long long* s_warp) {
    int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    int n = *pb.n_tiles;
    int nb = (n + 1023) >> 10;   // per-CTA sums (<= 16384 for max_tiles <= 2^24), scanned 256 at a time
    long long base = 0;
    for (int b0 = 0; b0 < nb; b0 += 256) {
        int b = b0 + tid;
        long long v = (b < nb) ? (long long)__ldcg(pb.block_sum + b) : 0, inc = v;
        for (int o = 1; o < 32; o <<= 1) {
            long long u = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += u;
        }
        __syncthreads();
        if (lane == 31) s_warp[wid] = inc;
        __syncthreads();
        long long woff = 0, total = 0;
        for (int i = 0; i < 8; ++i) { if (i < wid) woff += s_warp[i]; total += s_warp[i]; }
        if (b < nb) pb.block_base[b] = base + woff + inc - v;
        base += total;
    }
    if (tid == 0) {
        PlanStats* st = pb.stats;
        st->n_footprint = base;
        st->n_tiles = n;
        if (out_capacity >= 0 && base > out_capacity) plan_overflow(pb, 4);
        const int sc = *pb.slow_count;              // plan_members_kernel (the last to push) ran before this kernel
        *pb.slow_plan = sc < pb.max_tiles ? sc : pb.max_tiles;
    }
}

// 256 threads per CTA (so that a CTA fits beside the resample kernel's CTAs), 4 consecutive tiles per thread.
__global__ void __launch_bounds__(256) plan_offsets_kernel(PlanBuffers pb, long long out_capacity) {
    __shared__ int s_warp[8];
    __shared__ long long s_warp64[8];
    __shared__ int s_last;
    int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    int n = *pb.n_tiles;
    int i0 = blockIdx.x * 1024 + 4 * tid;       // this thread's 4 consecutive tiles (arrays are 256-byte aligned)
    if (blockIdx.x * 1024 < n) {
        int4 c4 = make_int4(0, 0, 0, 0);
        uchar4 k4 = make_uchar4(255, 255, 255, 255);
        if (i0 + 3 < n) {
            c4 = *reinterpret_cast<const int4*>(pb.tile_count + i0);
            k4 = *reinterpret_cast<const uchar4*>(pb.tile_cls + i0);
        } else {
            if (i0 < n) { c4.x = pb.tile_count[i0]; k4.x = pb.tile_cls[i0]; }
            if (i0 + 1 < n) { c4.y = pb.tile_count[i0 + 1]; k4.y = pb.tile_cls[i0 + 1]; }
            if (i0 + 2 < n) { c4.z = pb.tile_count[i0 + 2]; k4.z = pb.tile_cls[i0 + 2]; }
        }
        int c = c4.x + c4.y + c4.z + c4.w, inc = c;
        for (int o = 1; o < 32; o <<= 1) {
            int v = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += v;
        }
        if (lane == 31) s_warp[wid] = inc;
        int n_in = (k4.x == TC_INSIDE) + (k4.y == TC_INSIDE) + (k4.z == TC_INSIDE) + (k4.w == TC_INSIDE);
        int n_bo = (k4.x == TC_BORDER) + (k4.y == TC_BORDER) + (k4.z == TC_BORDER) + (k4.w == TC_BORDER);
        int n_ex = (k4.x == TC_EXACT) + (k4.y == TC_EXACT) + (k4.z == TC_EXACT) + (k4.w == TC_EXACT);
        int n_em = (k4.x == TC_EMPTY) + (k4.y == TC_EMPTY) + (k4.z == TC_EMPTY) + (k4.w == TC_EMPTY);
        n_in = __reduce_add_sync(0xffffffffu, n_in); n_bo = __reduce_add_sync(0xffffffffu, n_bo);
        n_ex = __reduce_add_sync(0xffffffffu, n_ex); n_em = __reduce_add_sync(0xffffffffu, n_em);
        if (lane == 0) {
            PlanStats* st = pb.stats;
            if (n_in) atomicAdd((unsigned long long*)&st->n_inside, (unsigned long long)n_in);
            if (n_bo) atomicAdd((unsigned long long*)&st->n_border, (unsigned long long)n_bo);
            if (n_ex) atomicAdd((unsigned long long*)&st->n_exact, (unsigned long long)n_ex);
            if (n_em) atomicAdd((unsigned long long*)&st->n_empty, (unsigned long long)n_em);
        }
        __syncthreads();
        int woff = 0, tot = 0;
        for (int i = 0; i < 8; ++i) { if (i < wid) woff += s_warp[i]; tot += s_warp[i]; }
        if (tid == 0) pb.block_sum[blockIdx.x] = tot;
        int ex = woff + inc - c;
        if (i0 + 3 < n) {
            *reinterpret_cast<int4*>(pb.tile_offset + i0) = make_int4(ex, ex + c4.x, ex + c4.x + c4.y, ex + c4.x + c4.y + c4.z);
        } else {
            if (i0 < n) pb.tile_offset[i0] = ex;
            if (i0 + 1 < n) pb.tile_offset[i0 + 1] = ex + c4.x;
            if (i0 + 2 < n) pb.tile_offset[i0 + 2] = ex + c4.x + c4.y;
        }
    }
    // the last CTA to arrive scans the per-CTA sums (block_base) and closes the statistics
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = (atomicAdd(pb.ticket, 1u) == gridDim.x - 1);
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    offsets_final_body(pb, out_capacity, s_warp64);
    if (tid == 0) *pb.ticket = 0u;
}

// Re-check of the caller's output capacity when a cached plan is reused (the scan did it when the plan was built).
__global__ void plan_check_capacity_kernel(PlanBuffers pb, long long out_capacity) {
    if (threadIdx.x == 0 && blockIdx.x == 0 && pb.stats->n_footprint > out_capacity) plan_overflow(pb, 4);
}

// *fetched = latch, latch = 0 (one atomic exchange: bits ORed in by kernels still running on other streams are kept
// for the next read).
__global__ void plan_latch_fetch_kernel(int* latch, int* fetched) {
    if (threadIdx.x == 0 && blockIdx.x == 0) *fetched = atomicExch(latch, 0);
}

__device__ __forceinline__ long long tile_out_offset(const PlanBuffers& pb, int t) {
    return pb.block_base[t >> 10] + pb.tile_offset[t];
}

// ------------------------------------------------------------------------------------ explicit list
// Expands the range plan into the ascending int64 footprint list (A1's explicit form).
__global__ void __launch_bounds__(256) plan_write_indices_kernel(PlanBuffers pb, long long* idx_out, long long capacity) {
    __shared__ unsigned s_mask[32];
    __shared__ int s_pref[33];
    int tid = threadIdx.x;
    int n = *pb.n_tiles;
    for (int t = blockIdx.x; t < n; t += gridDim.x) {
        int cls = pb.tile_cls[t];
        if (cls == TC_EMPTY) continue;
        long long base = pb.tile_id[t] << 10, off = tile_out_offset(pb, t);
        if (cls == TC_INSIDE) {
            for (int q = 0; q < 4; ++q) {
                int m = q * 256 + tid;
                if (off + m < capacity) idx_out[off + m] = base + m;
            }
        } else {
            __syncthreads();
            if (tid < 32) s_mask[tid] = pb.masks[(size_t)pb.rec[t].mask_slot * 32 + tid];
            __syncthreads();
            if (tid == 0) {
                int a = 0;
                for (int i = 0; i < 32; ++i) { s_pref[i] = a; a += __popc(s_mask[i]); }
                s_pref[32] = a;
            }
            __syncthreads();
            for (int q = 0; q < 4; ++q) {
                int m = q * 256 + tid;
                unsigned wd = s_mask[m >> 5];
                if ((wd >> (m & 31)) & 1u) {
                    long long pos = off + s_pref[m >> 5] + __popc(wd & ((1u << (m & 31)) - 1u));
                    if (pos < capacity) idx_out[pos] = base + m;
                }
            }
        }
    }
}
