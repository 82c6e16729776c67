// resample_unit.cuh -- A2..A5 (+A6) fused, bilinear or Lanczos-3, with IMAGE-ALIGNED work units: the second generation of the
// staged kernel.
//
// Why: a 32 x 32-pixel HEALPix tile is a diamond in the image, so the bounding box the tile kernel (resample_fast.cuh)
// stages holds 3.5 source pixels per output pixel, and its shape changes over the sky (polar-cap tiles are taller
// than wide).  Everything that scales with staged pixels -- L2 -> shared-memory traffic (the tile kernel runs at 86 % of
// the ~6300 B/clk L2 cap), TMA writes, the calibration pass -- is paid 3.5 times per output.  Here the unit of work is a
// RECTANGLE OF THE IMAGE (RW x RH source cells, e.g. 64 x 32): it owns the 4 x 4-pixel HEALPix sub-blocks (16
// consecutive nested indices = 64 contiguous output bytes) whose centre falls into it, and stages its rectangle plus
// the sub-blocks' overhang (3-4 cells) and the taps: 1.9 source pixels per output, ONE box shape for the whole frame
// (one TMA descriptor per array), the same shape at every pointing.
//
//   plan_units_kernel      (plan time) one warp per tile: unit of each of the tile's 64 sub-blocks from the tile cubic
//                          at the sub-block centre; per (unit, tile) one SEGMENT record {tile, 64-bit sub-block mask};
//                          sub-blocks whose pixels would leave their unit's box go to the stray list
//   resample_unit_kernel   persistent CTAs, 8 consumer warps + 2 producer warps, 2 stages; producer: TMA boxes, segment
//                          records (tile polynomials, output offsets, coadd slots, membership masks of border tiles),
//                          sub-block work list; consumers: calibrate the box once in place (as the tile kernel), then every
//                          half-warp takes one sub-block at a time: exact tile cubic per pixel (coefficients cached in
//                          registers while the segment stays the same), 2 x 2 taps, 64-byte contiguous stores
//   resample_stray_kernel  the stray sub-blocks, per pixel in FP64 with taps from global memory (none found by the plan in
//                          normal geometries; Lanczos-3 units with masked AND bright pixels hand theirs over at run time)
// Tiles the plan classifies TC_EXACT (belt/cap ring, poles) or whose cubic does not fit the fixed-point split stay on
// the slow list of the general kernel, exactly as with the tile kernel.
#pragma once
#include "resample_fast.cuh"

#define UNIT_MAXSEG 16                 // segments (distinct tiles) per unit
#define UNIT_MAXSB 384                 // sub-blocks per unit
#define UNIT_BOXW 72                   // staged box width (cells); 72 = 8 mod 16: pitch 72 is bank-conflict free
#ifndef UNIT_CAP
#define UNIT_CAP 3072                  // staged source pixels per stage (box width x box rows)
#endif
#ifndef UNIT_STAGES0
#define UNIT_STAGES0 2                  // stages with raw masters (14 B per staged pixel)
#endif

struct UnitGeom {
    int RW, RH;                        // cells owned by a unit
    int Mx, My;                        // overhang of a sub-block's pixels beyond its centre's cell (cells)
    int x_off, y_off;                  // unit (i, j) owns cells [x_off + i RW, + RW) x [y_off + j RH, + RH)
    int nux, nuy;
    int BW, BH;                        // staged box: cells [x0 - Mx - tl, ...) , BW x BH (BW % 8 == 0, origin % 8 == 0)
    int tl, tr;
    int max_stray;
    int chk_shrink;                    // ARGUS_DEBUG_BOUNDS self-test: the check pretends the box is this much narrower
};

struct __align__(16) UnitSeg {         // one (unit, tile) pair
    int t;                             // tile index in the plan
    unsigned mask_lo, mask_hi;         // sub-blocks of the tile owned by the unit (bit = Morton index of the 4 x 4 block)
    int pad;
};

struct UnitBuffers {
    int* nseg;                         // [n_units]
    UnitSeg* seg;                      // [n_units][UNIT_MAXSEG]
    int* stray_count;                  // device scalar: strays found by the plan
    int* stray_rt;                     // device scalar: sub-blocks handed over at run time (Lanczos-3: masked + bright boxes)
    int* stray_list;                   // [2 max_stray]  tile * 64 + sub-block; run-time entries from max_stray on
};

// Source position (2^-24 px relative to the record's integer base) of the point with doubled centred offsets (s, t):
// exact integer linear part + FP32 cubic remainder (common.cuh, FastRec).
__device__ __forceinline__ void unit_eval(const FastRec& r, int s, int t, int& xf, int& yf) {
    const float S = (float)s * 0.03125f, T = (float)t * 0.03125f;
    const float* px = r.px;
    const float* py = r.py;
    const float Ax = fmaf(S, fmaf(S, fmaf(S, px[6], px[3]), px[1]), px[0]), Bx = fmaf(S, fmaf(S, px[7], px[4]), px[2]), Cx = fmaf(S, px[8], px[5]);
    const float Ay = fmaf(S, fmaf(S, fmaf(S, py[6], py[3]), py[1]), py[0]), By = fmaf(S, fmaf(S, py[7], py[4]), py[2]), Cy = fmaf(S, py[8], py[5]);
    xf = r.c0x + r.ax * s + r.bx * t + __float_as_int(fmaf(T, fmaf(T, fmaf(T, px[9], Cx), Bx), Ax));
    yf = r.c0y + r.ay * s + r.by * t + __float_as_int(fmaf(T, fmaf(T, fmaf(T, py[9], Cy), By), Ay));
}

__device__ __forceinline__ int floor_div(int a, int b) { return (a >= 0) ? a / b : -((-a + b - 1) / b); }

// ------------------------------------------------------------------------------------------- plan side
// One warp per tile.  nseg and stray_count (one allocation) must be zero on entry (memset on the plan's stream).
__global__ void __launch_bounds__(256) plan_units_kernel(PlanBuffers pb, UnitGeom g, UnitBuffers ub) {
    __shared__ FastRec s_rec[8];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int n_tiles = *pb.n_tiles;
    for (int t = blockIdx.x * 8 + wid; t < n_tiles; t += gridDim.x * 8) {
        const int cls = pb.frec[t].cls;
        if (cls != TC_INSIDE && cls != TC_BORDER) continue;        // warp-uniform
        __syncwarp();
        if (lane < 10) reinterpret_cast<float4*>(&s_rec[wid])[lane] = __ldg(reinterpret_cast<const float4*>(pb.frec + t) + lane);
        __syncwarp();
        const FastRec& r = s_rec[wid];
        int key[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int sb = lane + 32 * h;
            const int a = (int)compact_even_bits((unsigned)sb), b = (int)compact_even_bits((unsigned)sb >> 1);
            key[h] = -1;
            bool member = true;
            if (cls == TC_BORDER) member = ((pb.masks[(size_t)r.mask_slot * 32 + (sb >> 1)] >> (16 * (sb & 1))) & 0xffffu) != 0;
            if (member) {
                int xf, yf;
                unit_eval(r, 8 * a - 28, 8 * b - 28, xf, yf);      // centre of the sub-block: u = 4 a + 1.5
                const int cx = r.X0 + (xf >> FAST_FRAC_BITS), cy = r.Y0 + (yf >> FAST_FRAC_BITS);
                const int i = floor_div(cx - g.x_off, g.RW), j = floor_div(cy - g.y_off, g.RH);
                bool ok = i >= 0 && i < g.nux && j >= 0 && j < g.nuy;
                // extent of the sub-block's pixels about its centre: the corner pixels are 3 half-pixel steps away in s and
                // in t; linear part exact, + 2^-6 px for the cubic's variation over 1.5 pixels (< 4e-3 px) and rounding
                const long long exl = 3ll * (llabs((long long)r.ax) + llabs((long long)r.bx)) + (1 << 18);
                const long long eyl = 3ll * (llabs((long long)r.ay) + llabs((long long)r.by)) + (1 << 18);
                const long long xc = ((long long)r.X0 << FAST_FRAC_BITS) + xf, yc = ((long long)r.Y0 << FAST_FRAC_BITS) + yf;
                const long long x_lo = (long long)(g.x_off + i * g.RW - g.Mx) << FAST_FRAC_BITS, x_hi = (long long)(g.x_off + (i + 1) * g.RW + g.Mx) << FAST_FRAC_BITS;
                const long long y_lo = (long long)(g.y_off + j * g.RH - g.My) << FAST_FRAC_BITS, y_hi = (long long)(g.y_off + (j + 1) * g.RH + g.My) << FAST_FRAC_BITS;
                ok = ok && xc - exl >= x_lo && xc + exl < x_hi && yc - eyl >= y_lo && yc + eyl < y_hi;
                key[h] = ok ? j * g.nux + i : -2;
            }
        }
        // strays (normally none)
#pragma unroll
        for (int h = 0; h < 2; ++h)
            if (key[h] == -2) {
                const int s = atomicAdd(ub.stray_count, 1);
                if (s < g.max_stray) ub.stray_list[s] = t * 64 + lane + 32 * h;
                else plan_overflow(pb, 2);
            }
        // one segment per distinct unit among the 64 sub-blocks: found one after the other (warp votes), appended by
        // different lanes at once (the atomics' latencies overlap)
        unsigned long long todo = (unsigned long long)__ballot_sync(0xffffffffu, key[0] >= 0) |
                                  ((unsigned long long)__ballot_sync(0xffffffffu, key[1] >= 0) << 32);
        int my_unit = -1, n_found = 0;
        unsigned my_lo = 0, my_hi = 0;
        while (todo) {
            const int bit = __ffsll((long long)todo) - 1;
            const int k0 = __shfl_sync(0xffffffffu, key[0], bit & 31), k1 = __shfl_sync(0xffffffffu, key[1], bit & 31);
            const int unit = (bit >> 5) ? k1 : k0;
            const unsigned m_lo = __ballot_sync(0xffffffffu, key[0] == unit), m_hi = __ballot_sync(0xffffffffu, key[1] == unit);
            todo &= ~((unsigned long long)m_lo | ((unsigned long long)m_hi << 32));
            if (lane == (n_found & 31)) {
                if (n_found < 32) { my_unit = unit; my_lo = m_lo; my_hi = m_hi; }
            }
            ++n_found;                                              // (a tile meets at most ~10 units; 32 is out of reach)
        }
        if (my_unit >= 0) {
            const int k = atomicAdd(ub.nseg + my_unit, 1);
            if (k < UNIT_MAXSEG) {
                UnitSeg sg;
                sg.t = t; sg.mask_lo = my_lo; sg.mask_hi = my_hi; sg.pad = 0;
                ub.seg[(size_t)my_unit * UNIT_MAXSEG + k] = sg;
            } else {                                                // more tiles than a unit can hold: its sub-blocks become strays
                unsigned long long m = (unsigned long long)my_lo | ((unsigned long long)my_hi << 32);
                while (m) {
                    const int sb = __ffsll((long long)m) - 1;
                    m &= m - 1;
                    const int sidx = atomicAdd(ub.stray_count, 1);
                    if (sidx < g.max_stray) ub.stray_list[sidx] = t * 64 + sb;
                    else plan_overflow(pb, 2);
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------- shared memory
// MASTERS: 0 = raw u16 + bias, dark, flat f32 (14 B per staged pixel), 1 = raw + offset, gain f32 (10 B),
// 2 = raw + offset, gain binary16 (6 B).
template <int MASTERS> struct UnitCfg {
    static constexpr int NARR = MASTERS == 0 ? 4 : 3;
    static constexpr int ES = MASTERS == 2 ? 2 : 4;                       // bytes per master element
    static constexpr int PX_BYTES = 2 + (NARR - 1) * ES;
    static constexpr int STAGE_BYTES = UNIT_CAP * PX_BYTES;
    static constexpr int STAGES = MASTERS == 2 ? 3 : (MASTERS == 0 ? UNIT_STAGES0 : 2);                   // 43 / 30 / 18 KB per stage: two CTAs per SM
};

struct __align__(16) UnitSegD {
    FastRec r;            // the tile's record (polynomial, integer bases, class, mask slot)
    long long off;        // output position of the tile's first pixel
    long long cslot;      // coadd slot of the tile's first pixel, -1 = tile absent from the layout
    int kofs;             // (Y0 - gy0) * pitch + (X0 - gx0)
    int mb;               // row of the border tables, -1 for inside tiles
    int pad[2];           // [0] = tile index in the plan
};
#define UNIT_PREFETCH 0                // L2 prefetch distance of the box loads in units of one CTA; 0 = off (measured: 3 is 7 % slower)
#define UNIT_PRODUCERS 2                // producer warps: the per-unit chain (records, offsets, work list) is a chain of latencies;
                                        // warp p prepares the CTA's units number p, p + PRODUCERS, ... (the kernel was producer-bound with one)
#define UNIT_THREADS (RF_CONSUMERS + 32 * UNIT_PRODUCERS)
#define UNIT_NDESC 4                   // descriptors are prepared up to three units ahead of the stage they describe
#define UNIT_MAXBORDER 6               // border-tile tables per unit (more: membership straight from global memory)
struct __align__(16) UnitDesc {
    int gx0, gy0, pad2, pad3;             // origin of the staged box (debug bounds check)
    int n_seg, n_sb, pad0, pad1;          // n_seg < 0: end of work; pad0 / pad1 = bit sets of the border segments / of segments absent from the coadd layout
    UnitSegD seg[UNIT_MAXSEG];
    unsigned sb[UNIT_MAXSB];              // work list, grouped by segment: segment << 12 | sub-block << 6 | a << 3 | b
    unsigned bmask[UNIT_MAXBORDER][32];   // border tiles: membership bits and exclusive prefix of their popcounts
    int bpref[UNIT_MAXBORDER][32];
};
template <int MASTERS>
struct __align__(128) UnitSmem {
    unsigned char stage[UnitCfg<MASTERS>::STAGES][UnitCfg<MASTERS>::STAGE_BYTES];
    UnitDesc desc[UNIT_NDESC];
    unsigned long long full[UNIT_NDESC];                     // descriptor written and TMA bytes landed
    unsigned long long empty[UnitCfg<MASTERS>::STAGES];      // all consumers are done with the stage
    unsigned long long dfree[UNIT_NDESC];                    // all consumers are done with the descriptor
};

struct UnitMaps { CUtensorMap m[4]; };    // raw, then the masters in stage order

__device__ __forceinline__ float calib_unit_pre(unsigned magic_r, float off, float g, float sat_f) {
    const float rf = __uint_as_float(magic_r) - 8388608.0f;
    const float c = (rf - off) * g;                                        // R-M4; NaN gain (invalid, off-frame) -> NaN
    return (rf < sat_f && fabsf(c) < INFINITY) ? c : nanf_();
}

// ------------------------------------------------------------------------------------------- the kernel
// 80 registers (no spills): two CTAs use 51 K of the SM's 64 K registers, the plan kernels of the next frame fit beside them
// (ARGUS_OPT_PLAN_OVERLAP)
#ifndef UNIT_MAXREG
#define UNIT_MAXREG 80
#endif
#define UNIT_BOUNDS __maxnreg__(UNIT_MAXREG)
template <bool COADD, int KERNEL, int MASTERS>
__global__ void UNIT_BOUNDS
    resample_unit_kernel(const __grid_constant__ UnitMaps maps, PlanBuffers pb, UnitBuffers ub, UnitGeom g, FrameArgs f, float w_min,
                         float* __restrict__ value_out, float* __restrict__ weight_out, long long out_cap, CoaddArgs ca) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    typedef UnitCfg<MASTERS> Cfg;
    constexpr int NI = (UNIT_CAP / 4 + RF_CONSUMERS - 1) / RF_CONSUMERS;
    UnitSmem<MASTERS>& sm = *reinterpret_cast<UnitSmem<MASTERS>*>(smem_raw);
    const int tid = threadIdx.x;
    const int n_units = g.nux * g.nuy;
    const int pitch = fast_cal_pitch(g.BW);

    if (tid == 0) {
        for (int i = 0; i < UNIT_NDESC; ++i) { mbar_init(&sm.full[i], 1); mbar_init(&sm.dfree[i], RF_CONSUMERS); }
        for (int i = 0; i < Cfg::STAGES; ++i) mbar_init(&sm.empty[i], RF_CONSUMERS);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (tid >= RF_CONSUMERS) {
        // ================================================================ producer warp
        const int lane = tid & 31, pw = (tid - RF_CONSUMERS) >> 5;      // producer warp pw of UNIT_PRODUCERS
        int issued = 0;                                                 // sequence number of the CTA's non-empty units
        int u_n = blockIdx.x, nseg_n = 0;
        UnitSeg sg_n = {0, 0u, 0u, 0};
        if (u_n < n_units) {
            nseg_n = min(__ldg(ub.nseg + u_n), UNIT_MAXSEG);
            if (lane < nseg_n) sg_n = ub.seg[(size_t)u_n * UNIT_MAXSEG + lane];
        }
        for (;;) {
            const int u = u_n, nseg = nseg_n;
            const UnitSeg sg = sg_n;
            const bool last = u >= n_units;
            u_n = u + gridDim.x;
            nseg_n = 0;
            if (u_n < n_units) {
                nseg_n = min(__ldg(ub.nseg + u_n), UNIT_MAXSEG);
                if (lane < nseg_n) sg_n = ub.seg[(size_t)u_n * UNIT_MAXSEG + lane];
            }
            if (!last && nseg == 0) continue;
            if (issued % UNIT_PRODUCERS != pw) {                        // another producer warp's unit
                if (last) break;
                ++issued;
                continue;
            }
            const int slot = issued % Cfg::STAGES, ds = issued % UNIT_NDESC;
            // descriptor slot free: the consumers are done with the unit that used it UNIT_NDESC units ago
            if (issued >= UNIT_NDESC) mbar_wait(&sm.dfree[ds], (unsigned)((issued / UNIT_NDESC - 1) & 1));
            UnitDesc& d = sm.desc[ds];
            if (last) {
                if (lane == 0) { d.n_seg = -1; mbar_arrive(&sm.full[ds]); }
                break;
            }
            const int ui = u % g.nux, uj = u / g.nux;
            const int gx0 = g.x_off + ui * g.RW - g.Mx - g.tl, gy0 = g.y_off + uj * g.RH - g.My - g.tl;
            // The kernel is bound by the latency of its box loads (two stages in flight per CTA are less than the
            // bandwidth-delay product): the boxes of the unit UNIT_PREFETCH steps ahead are pulled into L2 now, so that its
            // TMA copies find them there.
            {
                const int up = u + UNIT_PREFETCH * (int)gridDim.x;
                if (UNIT_PREFETCH > 0 && lane < Cfg::NARR && up < n_units && __ldg(ub.nseg + up) > 0) {
                    const int pi = up % g.nux, pj = up / g.nux;
                    tma_prefetch_2d(&maps.m[lane], g.x_off + pi * g.RW - g.Mx - g.tl, g.y_off + pj * g.RH - g.My - g.tl);
                }
            }
            // tile records of the segments: lane l copies half (5 x 16 B) of segment l / 2's record
            {
                const int t_l = __shfl_sync(0xffffffffu, sg.t, lane >> 1);
                if ((lane >> 1) < nseg) {
                    const float4* src = reinterpret_cast<const float4*>(pb.frec + t_l) + 5 * (lane & 1);
                    float4* dst = reinterpret_cast<float4*>(&d.seg[lane >> 1].r) + 5 * (lane & 1);
                    float4 v[5];
#pragma unroll
                    for (int k = 0; k < 5; ++k) v[k] = __ldg(src + k);
#pragma unroll
                    for (int k = 0; k < 5; ++k) dst[k] = v[k];
                }
            }
            long long off_l = 0, cs_l = -1;
            if (lane < nseg) {
                off_l = tile_out_offset(pb, sg.t);
                if (COADD) {
                    cs_l = pb.cslot[sg.t];                      // coadd_slots_kernel, once per call
#ifndef ARGUS_NO_COADD_PREFETCH
                    // the segment's tile accumulators towards L2 ahead of the consumers' read-modify-write (as in the tile kernel;
                    // the units that share a tile find it there already)
                    if (cs_l >= 0 && ((((unsigned long long)ca.sum | (unsigned long long)ca.wsum) & 15ull) == 0ull)) {   // (the API asks for 4-byte alignment only)
                        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" :: "l"(ca.sum + cs_l), "r"(ARGUS_TILE_PIX * 4) : "memory");
                        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" :: "l"(ca.wsum + cs_l), "r"(ARGUS_TILE_PIX * 4) : "memory");
                    }
#endif
                }
            }
            __syncwarp();
            int cls_l = 0, mslot_l = 0;
            if (lane < nseg) {
                UnitSegD& sd = d.seg[lane];
                cls_l = sd.r.cls; mslot_l = sd.r.mask_slot;
                sd.off = off_l; sd.cslot = cs_l; sd.pad[0] = sg.t;
                sd.kofs = (sd.r.Y0 - gy0) * pitch + (sd.r.X0 - gx0);
            }
            const unsigned border = __ballot_sync(0xffffffffu, lane < nseg && cls_l == TC_BORDER);
            if (lane < nseg) {
                const int row = __popc(border & ((1u << lane) - 1u));
                d.seg[lane].mb = (cls_l != TC_BORDER) ? -1 : (row < UNIT_MAXBORDER ? row : -2 - mslot_l);   // <= -2: masks from global memory
            }
            // work list, grouped by segment: every lane places two bit positions of each segment's mask
            const unsigned long long mk = (lane < nseg) ? ((unsigned long long)sg.mask_lo | ((unsigned long long)sg.mask_hi << 32)) : 0ull;
            const int cnt = __popcll(mk);
            int inc = cnt;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += y;
            }
            const int total = __shfl_sync(0xffffffffu, inc, 31);
            const int la = (int)compact_even_bits((unsigned)lane), lb = (int)compact_even_bits((unsigned)lane >> 1);   // lane = sub-block & 31
            for (int sgi = 0; sgi < nseg; ++sgi) {
                const unsigned m_lo = __shfl_sync(0xffffffffu, (unsigned)mk, sgi), m_hi = __shfl_sync(0xffffffffu, (unsigned)(mk >> 32), sgi);
                const int base = __shfl_sync(0xffffffffu, inc - cnt, sgi);
                const unsigned below = (1u << lane) - 1u;
                if ((m_lo >> lane) & 1u) {
                    const int pos = base + __popc(m_lo & below);
                    if (pos < UNIT_MAXSB) d.sb[pos] = (unsigned)(sgi << 12) | (unsigned)(lane << 6) | (unsigned)(la << 3) | (unsigned)lb;
                }
                if ((m_hi >> lane) & 1u) {                          // sub-block lane + 32: b gains bit 2 (32 = bit 5 = iy bit 2)
                    const int pos = base + __popc(m_lo) + __popc(m_hi & below);
                    if (pos < UNIT_MAXSB) d.sb[pos] = (unsigned)(sgi << 12) | (unsigned)((lane + 32) << 6) | (unsigned)(la << 3) | (unsigned)(lb + 4);
                }
            }
            if (total > UNIT_MAXSB && lane == 0) plan_overflow(pb, 2);     // geometry guard (host sizes units for < 0.55 MAXSB)
            // border tiles: membership words + exclusive prefix
            for (unsigned bm = border; bm; bm &= bm - 1) {
                const int sgi = __ffs(bm) - 1, row = __popc(border & ((1u << sgi) - 1u));
                if (row >= UNIT_MAXBORDER) break;
                const int ms = __shfl_sync(0xffffffffu, mslot_l, sgi);
                const unsigned w = pb.masks[(size_t)ms * 32 + lane];
                const int c = __popc(w);
                int ic = c;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int y = __shfl_up_sync(0xffffffffu, ic, o);
                    if (lane >= o) ic += y;
                }
                d.bmask[row][lane] = w;
                d.bpref[row][lane] = ic - c;
            }
            const unsigned absent = __ballot_sync(0xffffffffu, COADD && lane < nseg && cs_l < 0);
            if (lane == 0) { d.n_seg = nseg; d.n_sb = min(total, UNIT_MAXSB); d.pad0 = (int)border; d.pad1 = (int)absent; d.gx0 = gx0; d.gy0 = gy0; }
            __syncwarp();
            // stage free: every consumer is done with the unit that used it STAGES units ago; then the bulk copies
            if (issued >= Cfg::STAGES) mbar_wait(&sm.empty[slot], (unsigned)((issued / Cfg::STAGES - 1) & 1));
            if (lane == 0) {
                unsigned char* st = sm.stage[slot];
                tma_load_2d(st, &maps.m[0], gx0, gy0, &sm.full[ds]);
#pragma unroll
                for (int a = 1; a < Cfg::NARR; ++a)
                    tma_load_2d(st + UNIT_CAP * 2 + (a - 1) * UNIT_CAP * Cfg::ES, &maps.m[a], gx0, gy0, &sm.full[ds]);
                mbar_arrive_expect_tx(&sm.full[ds], (unsigned)(g.BW * g.BH * Cfg::PX_BYTES));
            }
            ++issued;
        }
        return;
    }

    // ==================================================================== consumer warps
    const int gt = tid;
    const int half = gt >> 4;                                   // 16 sub-block slots per pass, one per half-warp
    const int q = gt & 15;                                      // pixel of the sub-block (Morton order)
    const int du = (int)compact_even_bits((unsigned)q), dv = (int)compact_even_bits((unsigned)q >> 1);
    const unsigned fmin_bits = __float_as_uint(f.flat_min), frange = 0x7f800000u - fmin_bits;
    const float sat_f = (float)f.sat_adu, t_exp = f.t_exp;
    const int bw4 = g.BW >> 2, n4 = g.BH * bw4;
    const unsigned M = (1048576u + bw4 - 1) / bw4;              // exact division by bw4 for v < 2^14

    for (int it = 0;; ++it) {
        const int slot = it % Cfg::STAGES, ds = it % UNIT_NDESC;
        mbar_wait(&sm.full[ds], (unsigned)((it / UNIT_NDESC) & 1));
        const UnitDesc& d = sm.desc[ds];
        const int n_seg = d.n_seg;
        if (n_seg < 0) break;
        unsigned char* st = sm.stage[slot];
        float* cal = reinterpret_cast<float*>(st);
        // ---- A2: calibrate the staged box once (dense: item v <-> 4 pixels), registers -> barrier -> in place
        float4 o4[NI];
        int bad = 0, big = 0;
#pragma unroll
        for (int j = 0; j < NI; ++j) {
            const int v = gt + RF_CONSUMERS * j;
            if (v < n4) {
                const uint2 rw = reinterpret_cast<const uint2*>(st)[v];
                const unsigned m0 = __byte_perm(rw.x, 0x4B000000u, 0x7610), m1 = __byte_perm(rw.x, 0x4B000000u, 0x7632);
                const unsigned m2 = __byte_perm(rw.y, 0x4B000000u, 0x7610), m3 = __byte_perm(rw.y, 0x4B000000u, 0x7632);
                if (MASTERS == 0) {
                    const float4 b = reinterpret_cast<const float4*>(st + UNIT_CAP * 2)[v];
                    const float4 dk = reinterpret_cast<const float4*>(st + UNIT_CAP * 6)[v];
                    const float4 fl = reinterpret_cast<const float4*>(st + UNIT_CAP * 10)[v];
                    int bad4 = 0;                    // (the NaN test below covers both kinds of masters)
                    o4[j] = calib_fast4<KERNEL == 1>(rw, b, dk, fl, t_exp, sat_f, fmin_bits, frange, bad4);
                } else {
                    float4 of, gn;
                    if (MASTERS == 1) {
                        of = reinterpret_cast<const float4*>(st + UNIT_CAP * 2)[v];
                        gn = reinterpret_cast<const float4*>(st + UNIT_CAP * 6)[v];
                    } else {
                        const uint2 ho = reinterpret_cast<const uint2*>(st + UNIT_CAP * 2)[v], hg = reinterpret_cast<const uint2*>(st + UNIT_CAP * 4)[v];
                        const float2 o01 = __half22float2(*reinterpret_cast<const __half2*>(&ho.x)), o23 = __half22float2(*reinterpret_cast<const __half2*>(&ho.y));
                        const float2 g01 = __half22float2(*reinterpret_cast<const __half2*>(&hg.x)), g23 = __half22float2(*reinterpret_cast<const __half2*>(&hg.y));
                        of = make_float4(o01.x, o01.y, o23.x, o23.y);
                        gn = make_float4(g01.x, g01.y, g23.x, g23.y);
                    }
                    o4[j].x = calib_unit_pre(m0, of.x, gn.x, sat_f);
                    o4[j].y = calib_unit_pre(m1, of.y, gn.y, sat_f);
                    o4[j].z = calib_unit_pre(m2, of.z, gn.z, sat_f);
                    o4[j].w = calib_unit_pre(m3, of.w, gn.w, sat_f);
                }
                bad |= (o4[j].x != o4[j].x) | (o4[j].y != o4[j].y) | (o4[j].z != o4[j].z) | (o4[j].w != o4[j].w);
                if (KERNEL == 1) big |= (fmaxf(fmaxf(fabsf(o4[j].x), fabsf(o4[j].y)), fmaxf(fabsf(o4[j].z), fabsf(o4[j].w))) > RF_LZ_BIG_ADU);
            }
        }
        const int any_bad = bar_sync_or<1>(bad);
        const int any_big = KERNEL == 1 ? bar_sync_or<1>(big) : 0;
#pragma unroll
        for (int j = 0; j < NI; ++j) {
            const int v = gt + RF_CONSUMERS * j;
            if (v < n4) {
                const int row = (int)(((unsigned)v * M) >> 20);
                *reinterpret_cast<float4*>(cal + row * pitch + 4 * (v - row * bw4)) = o4[j];
            }
        }
        bar_sync<1>();
        const int n_sb = d.n_sb;
        if (KERNEL == 1 && any_big && any_bad) {
            // Lanczos-3 with masked taps next to bright pixels (saturated star cores) needs FP64 weights and coordinates
            // (DESIGN.md 6.2): the unit's sub-blocks are handed to the stray kernel, which runs after this one.
            for (int e = gt; e < n_sb; e += RF_CONSUMERS) {
                const unsigned ent = d.sb[e];
                const int k = atomicAdd(ub.stray_rt, 1);
                if (k < g.max_stray) ub.stray_list[g.max_stray + k] = d.seg[ent >> 12].pad[0] * 64 + (int)((ent >> 6) & 63u);
                else plan_overflow(pb, 2);
            }
            mbar_arrive(&sm.empty[slot]);
            mbar_arrive(&sm.dfree[ds]);
            continue;
        }

        // ---- A3..A5: one sub-block per half-warp and pass; the segment's coefficients stay in registers
        int cur = -1;
        float px0 = 0, px1 = 0, px2 = 0, px3 = 0, px4 = 0, px5 = 0, px6 = 0, px7 = 0, px8 = 0, px9 = 0;
        float py0 = 0, py1 = 0, py2 = 0, py3 = 0, py4 = 0, py5 = 0, py6 = 0, py7 = 0, py8 = 0, py9 = 0;
        int c0x = 0, axi = 0, bxi = 0, c0y = 0, ayi = 0, byi = 0, mb = -1;
        const float* cb = cal;
        long long off = 0, cslot = -1;
        int dbg_x = 0, dbg_y = 0;
        (void)dbg_x; (void)dbg_y;
        const int sdu = 2 * du - 31, sdv = 2 * dv - 31;
#define UNIT_LOAD_SEG(SGI)                                                                                        \
    {                                                                                                             \
        const UnitSegD& sd = d.seg[SGI];                                                                          \
        px0 = sd.r.px[0]; px1 = sd.r.px[1]; px2 = sd.r.px[2]; px3 = sd.r.px[3]; px4 = sd.r.px[4];                 \
        px5 = sd.r.px[5]; px6 = sd.r.px[6]; px7 = sd.r.px[7]; px8 = sd.r.px[8]; px9 = sd.r.px[9];                 \
        py0 = sd.r.py[0]; py1 = sd.r.py[1]; py2 = sd.r.py[2]; py3 = sd.r.py[3]; py4 = sd.r.py[4];                 \
        py5 = sd.r.py[5]; py6 = sd.r.py[6]; py7 = sd.r.py[7]; py8 = sd.r.py[8]; py9 = sd.r.py[9];                 \
        c0x = sd.r.c0x; axi = sd.r.ax; bxi = sd.r.bx; c0y = sd.r.c0y; ayi = sd.r.ay; byi = sd.r.by;               \
        cb = cal + sd.kofs; mb = sd.mb; off = sd.off; cslot = sd.cslot;                                           \
        dbg_x = sd.r.X0 - d.gx0; dbg_y = sd.r.Y0 - d.gy0;                                                         \
        cur = SGI;                                                                                                \
    }
#define UNIT_POSITION(ENT)                                                                                        \
    const int s = 8 * (int)((ENT >> 3) & 7u) + sdu, t = 8 * (int)(ENT & 7u) + sdv;                                \
    const float S = (float)s * 0.03125f, T = (float)t * 0.03125f;                                                 \
    const float Ax = fmaf(S, fmaf(S, fmaf(S, px6, px3), px1), px0), Bx = fmaf(S, fmaf(S, px7, px4), px2), Cx = fmaf(S, px8, px5); \
    const float Ay = fmaf(S, fmaf(S, fmaf(S, py6, py3), py1), py0), By = fmaf(S, fmaf(S, py7, py4), py2), Cy = fmaf(S, py8, py5); \
    const int xf = c0x + axi * s + bxi * t + __float_as_int(fmaf(T, fmaf(T, fmaf(T, px9, Cx), Bx), Ax));           \
    const int yf = c0y + ayi * s + byi * t + __float_as_int(fmaf(T, fmaf(T, fmaf(T, py9, Cy), By), Ay));           \
    const float* a = cb + ((yf >> FAST_FRAC_BITS) * pitch + (xf >> FAST_FRAC_BITS));
        // a unit without border tiles and without a masked pixel in its box (nearly all): no membership, no weights
        if (!any_bad && d.pad0 == 0 && (!COADD || d.pad1 == 0)) {
            // eight threads per sub-block, two vertically adjacent pixels each (same column: the S-dependent Horner
            // coefficients are shared): in-block Morton indices q0 and q0 + 2
            const int oct = gt >> 3, i8 = gt & 7;
            const int q0 = (i8 & 1) | ((i8 >> 1) << 2);
            const int sdu2 = 2 * (i8 & 3) - 31, sdv2 = 4 * (i8 >> 2) - 31;
            float* vq = value_out + q0;
            float* wq = weight_out + q0;
            for (int e = oct; e < n_sb; e += RF_CONSUMERS / 8) {
                const unsigned ent = d.sb[e];
                const int sgi = (int)(ent >> 12);
                if (sgi != cur) UNIT_LOAD_SEG(sgi)                  // uniform over the eight threads
                // A6: the accumulator loads are issued before the position arithmetic, their latency hides under it
                float* sp = nullptr;
                float* wp = nullptr;
                float s_a0 = 0.f, s_a1 = 0.f, w_a0 = 0.f, w_a1 = 0.f;
                if (COADD) {
                    sp = ca.sum + cslot + ((ent >> 2) & 0x3f0u) + q0;
                    wp = ca.wsum + cslot + ((ent >> 2) & 0x3f0u) + q0;
                    s_a0 = sp[0]; s_a1 = sp[2]; w_a0 = wp[0]; w_a1 = wp[2];
                }
                const int s = 8 * (int)((ent >> 3) & 7u) + sdu2, t = 8 * (int)(ent & 7u) + sdv2;
                const float S = (float)s * 0.03125f, T0 = (float)t * 0.03125f, T1 = T0 + 0.0625f;
                const float Ax = fmaf(S, fmaf(S, fmaf(S, px6, px3), px1), px0), Bx = fmaf(S, fmaf(S, px7, px4), px2), Cx = fmaf(S, px8, px5);
                const float Ay = fmaf(S, fmaf(S, fmaf(S, py6, py3), py1), py0), By = fmaf(S, fmaf(S, py7, py4), py2), Cy = fmaf(S, py8, py5);
                const int lx = c0x + axi * s + bxi * t, ly = c0y + ayi * s + byi * t;
                const int xf0 = lx + __float_as_int(fmaf(T0, fmaf(T0, fmaf(T0, px9, Cx), Bx), Ax));
                const int yf0 = ly + __float_as_int(fmaf(T0, fmaf(T0, fmaf(T0, py9, Cy), By), Ay));
                const int xf1 = lx + 2 * bxi + __float_as_int(fmaf(T1, fmaf(T1, fmaf(T1, px9, Cx), Bx), Ax));
                const int yf1 = ly + 2 * byi + __float_as_int(fmaf(T1, fmaf(T1, fmaf(T1, py9, Cy), By), Ay));
                RF_CHECK_BOX(pb, dbg_x + (xf0 >> FAST_FRAC_BITS), dbg_y + (yf0 >> FAST_FRAC_BITS), g.tl, g.tr, g.BW - g.chk_shrink, g.BH)
                RF_CHECK_BOX(pb, dbg_x + (xf1 >> FAST_FRAC_BITS), dbg_y + (yf1 >> FAST_FRAC_BITS), g.tl, g.tr, g.BW - g.chk_shrink, g.BH)
                const float* a0 = cb + ((yf0 >> FAST_FRAC_BITS) * pitch + (xf0 >> FAST_FRAC_BITS));
                const float* a1 = cb + ((yf1 >> FAST_FRAC_BITS) * pitch + (xf1 >> FAST_FRAC_BITS));
                const float v0 = interp_clean<KERNEL>(a0, pitch, fast_frac(xf0), fast_frac(yf0));
                const float v1 = interp_clean<KERNEL>(a1, pitch, fast_frac(xf1), fast_frac(yf1));
                if (COADD) {        // footprint pixels are unique within a frame: plain read-modify-write, deterministic
                    sp[0] = s_a0 + v0; sp[2] = s_a1 + v1;
                    wp[0] = w_a0 + 1.0f; wp[2] = w_a1 + 1.0f;
                    continue;
                }
                const long long o = off + (long long)((ent >> 2) & 0x3f0u);      // 16 * sub-block
                if (o + 16 <= out_cap) {
                    vq[o] = v0; vq[o + 2] = v1;
                    wq[o] = 1.0f; wq[o + 2] = 1.0f;
                } else {
                    if (o + q0 < out_cap) { vq[o] = v0; wq[o] = 1.0f; }
                    if (o + q0 + 2 < out_cap) { vq[o + 2] = v1; wq[o + 2] = 1.0f; }
                }
            }
        } else {
            for (int e = half; e < n_sb; e += RF_CONSUMERS / 16) {
                const unsigned ent = d.sb[e];
                const int sgi = (int)(ent >> 12), sb = (int)(ent >> 6) & 63;
                if (sgi != cur) UNIT_LOAD_SEG(sgi)
                UNIT_POSITION(ent)
                const int m = 16 * sb + q;                          // Morton index of the pixel in its tile
                bool member = true;
                long long pos = m;
                if (mb >= 0) {
                    const unsigned wd = d.bmask[mb][sb >> 1];
                    const int bit = 16 * (sb & 1) + q;
                    member = (wd >> bit) & 1u;
                    pos = d.bpref[mb][sb >> 1] + __popc(wd & ((1u << bit) - 1u));
                } else if (mb <= -2) {                              // more border tiles in the unit than tables: global memory
                    const unsigned* mkp = pb.masks + (size_t)(-2 - mb) * 32;
                    const unsigned wd = mkp[sb >> 1];
                    const int bit = 16 * (sb & 1) + q;
                    member = (wd >> bit) & 1u;
                    pos = __popc(wd & ((1u << bit) - 1u));
                    for (int k = 0; k < (sb >> 1); ++k) pos += __popc(mkp[k]);
                }
                if (!member) continue;
                RF_CHECK_BOX(pb, dbg_x + (xf >> FAST_FRAC_BITS), dbg_y + (yf >> FAST_FRAC_BITS), g.tl, g.tr, g.BW - g.chk_shrink, g.BH)
                const float fx = fast_frac(xf), fy = fast_frac(yf);
                float val, wgt;
                if (!any_bad) { val = interp_clean<KERNEL>(a, pitch, fx, fy); wgt = 1.0f; }
                else interp_masked<KERNEL>(a, pitch, fx, fy, w_min, val, wgt);
                if (COADD) {
                    if (cslot >= 0) {
                        // footprint pixels are unique within a frame: plain read-modify-write, deterministic
                        float* sp = ca.sum + cslot + m;
                        float* wp = ca.wsum + cslot + m;
                        *sp = fmaf(wgt, val, *sp);
                        *wp += wgt;
                    } else if (ca.n_skipped) {
                        atomicAdd(ca.n_skipped, 1ull);
                    }
                } else if (off + pos < out_cap) {
                    value_out[off + pos] = val;
                    weight_out[off + pos] = wgt;
                }
            }
        }
#undef UNIT_LOAD_SEG
#undef UNIT_POSITION
        mbar_arrive(&sm.empty[slot]);
        mbar_arrive(&sm.dfree[ds]);
    }
}

// ------------------------------------------------------------------------------------------- strays
// Sub-blocks the unit kernel does not serve -- found by the plan (their pixels would leave the unit's box) or handed over at
// run time (Lanczos-3 next to masked + bright pixels) -- per pixel, exact FP64 coordinates, taps from global memory, FP64
// Lanczos weights.
template <int KERNEL, bool COADD>
__global__ void __launch_bounds__(256) resample_stray_kernel(DevWcs w, PlanBuffers pb, UnitBuffers ub, int max_stray, FrameArgs f,
                                                            float w_min, float* __restrict__ value_out, float* __restrict__ weight_out,
                                                            long long out_cap, CoaddArgs ca) {
    const int n0 = min(*ub.stray_count, max_stray), n1 = min(*ub.stray_rt, max_stray);
    for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < 16ll * (n0 + n1); i += (long long)gridDim.x * 256) {
        const long long e = i >> 4;
        const int ent = ub.stray_list[e < n0 ? e : max_stray + (e - n0)], t = ent >> 6, sb = ent & 63, q = (int)(i & 15);
        const int m = 16 * sb + q;
        const long long tile = pb.tile_id[t];
        long long pos = m;
        if (pb.tile_cls[t] == TC_BORDER) {
            const unsigned* mk = pb.masks + (size_t)pb.frec[t].mask_slot * 32;
            const unsigned wd = mk[m >> 5];
            if (!((wd >> (m & 31)) & 1u)) continue;
            pos = __popc(wd & ((1u << (m & 31)) - 1u));
            for (int k = 0; k < (m >> 5); ++k) pos += __popc(mk[k]);
        }
        int face, tx, ty;
        nest_to_xyf(tile, w.k - ARGUS_TILE_LOG2, face, tx, ty);
        const int u = (int)compact_even_bits((unsigned)m), v = (int)compact_even_bits((unsigned)m >> 1);
        double x, y;
        pixel_to_xy(w, face, tx * 32 + u, ty * 32 + v, x, y);
        const double flx = floor(x), fly = floor(y);
        GlobalTaps<true, KERNEL == 1> gt{&f, w.W, w.H};
        float val, wgt;
        if (KERNEL == 0) interp_bilinear_masked(gt, (int)flx, (int)fly, (float)(x - flx), (float)(y - fly), w_min, val, wgt);
        else interp_lanczos3_masked(gt, (int)flx, (int)fly, x - flx, y - fly, w_min, val, wgt);
        if (COADD) {
            const long long sl0 = pb.cslot[t];                       // coadd_slots_kernel
            if (sl0 >= 0) {
                ca.sum[sl0 + m] = fmaf(wgt, val, ca.sum[sl0 + m]);
                ca.wsum[sl0 + m] += wgt;
            } else if (ca.n_skipped) {
                atomicAdd(ca.n_skipped, 1ull);
            }
        } else {
            const long long o = tile_out_offset(pb, t) + pos;
            if (o < out_cap) { value_out[o] = val; weight_out[o] = wgt; }
        }
    }
}
