// argus_api.cu -- the C ABI declared in include/argus.h: validation, host-side frame constants (FP64),
// coarse cell selection, kernel launches.  Every step of the hot path runs in the kernels of
// plan.cuh / resample.cuh; nothing here touches pixel data.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/argus.h"
#include "plan_block.cuh"
#include "resample.cuh"
#include "resample_fast.cuh"
#include "resample_unit.cuh"
#include "segments.cuh"
#include "background.cuh"
#include "subtract.cuh"

#define ARGUS_VERSION_NUM 100
#define PLAN_SLOTS 3

struct argus_ctx {
    int device;
    int last_cuda;
    int sm_count;
    bool plan_cache;
    bool plan_valid;
    bool plan_full;       // the cached plan holds TileRec / FP64 coefficients for every tile (general kernel)
    int plan_fast_kernel; // interpolation kernel whose tap apron sized the fast kernel's boxes in the cached plan
    int plan_fast_cap;    // stage capacity those boxes were checked against (FastCfg<..>::CAP)
    bool lz_small_enabled;// ARGUS_OPT_FAST_PATH != 4
    bool lz_small;        // choose_path: every tile of this frame fits the small Lanczos-3 stage (FastCfg<1, 1>)
    argus_wcs key_wcs;
    int64_t key_W, key_H, key_nside;
    DevWcs dw;
    PlanBuffers pb;
    PlanStats* h_stats;   // pinned
    bool profile;
    int prof_n;           // calls recorded since the last read
    cudaEvent_t ev[256][4];   // plan begin / end (on the stream the plan ran on), resample begin / end (caller's stream)
    bool ev_plan[256];    // the call re-planned (ev[i][0] -> ev[i][1] is meaningful)
    // PLAN_SLOTS sets of plan scratch: with ARGUS_OPT_PLAN_OVERLAP the plan of a new WCS is built on a high-priority
    // side stream in the set whose last reader is oldest, so it runs underneath the previous frames' kernels (up to
    // PLAN_SLOTS - 1 frames ahead of them).
    PlanBuffers slot_pb[PLAN_SLOTS];
    void* slot_block[PLAN_SLOTS];
    int cur_slot;
    bool overlap;
    bool slot_used[PLAN_SLOTS];   // ev_free[s] has been recorded
    cudaStream_t side[2];     // plans of consecutive frames alternate between two side streams (two plans in flight)
    int side_next;
    cudaEvent_t ev_done[PLAN_SLOTS];   // plan of the slot complete (side stream)
    cudaEvent_t ev_free[PLAN_SLOTS];   // last kernel reading the slot complete (caller's stream)
    // TMA descriptors of the fast kernel, cached per (pointers, W, H)
    void* encode_fn;      // cuTensorMapEncodeTiled, resolved at first use (no link-time libcuda dependency)
    bool encode_tried;
    bool fast_enabled;    // ARGUS_OPT_FAST_PATH != 0
    int unit_margin;      // ARGUS_OPT_UNIT_MARGIN
    bool unit_forced;     // ARGUS_OPT_FAST_PATH == 3: units wherever their geometry allows (diagnostic)
    bool unit_enabled;    // ARGUS_OPT_FAST_PATH == 1 or 3: image-aligned work units (resample_unit.cuh) where the geometry allows
    bool fast_attr_set;
    bool unit_attr_set;
    bool plan_unit;       // the cached plan carries unit segment lists for plan_geom
    UnitGeom plan_geom;
    UnitBuffers slot_ub[PLAN_SLOTS];
    void* unit_block[PLAN_SLOTS];
    size_t unit_cap;      // units the unit scratch holds
    UnitMaps umaps;       // TMA descriptors of the unit kernel, cached per (pointers, W, H, box, masters format)
    const void* umaps_key[4];
    int64_t umaps_W, umaps_H;
    int umaps_bw, umaps_bh, umaps_fmt;
    FastMaps maps;
    const void* maps_key[4];
    int64_t maps_W, maps_H;
    int64_t n_launches;   // kernels launched through this context (diagnostics)
    bool auto_tiles;      // max_tiles = 0 at creation: the plan scratch is sized from (W, H, nside, pixel scale) at first use
    int64_t cap_tiles, cap_slots;   // capacity of the allocated scratch sets (0 = none yet)
    int* d_latch;         // [0] overflow bits of every asynchronous call since the last read, [1] the value last fetched
    int* h_latch;         // pinned copy of d_latch[1]
    // argus_resample_host: two sets of device staging buffers, upload / download streams
    struct HostBuf {
        uint16_t* raw; float* val; float* wgt;
        size_t cap_px, cap_n;
        // argus_reduce_frame_host: footprint list, binary16 segment data, low-resolution map
        long long* idx; uint16_t* seg16; size_t cap_prod;
        long long* mini_id; float* mini_val; float* mini_wgt; long long* n_mini; size_t cap_mini;
        cudaEvent_t up, run, down;
        bool used, down_used, ev_ok;
    } hb[2];
    int hb_next;
    cudaStream_t s_up, s_down;
    // argus_segment_products: head positions, look-back words ([0] ticket, [1] n_mini, [2..] one per head-scan CTA)
    struct SegScratch {
        long long* mini_start; size_t cap_mini;
        unsigned long long* ctl; size_t cap_ctas;
        long long* h_n;   // pinned
    } seg;
    bool seg_raster;      // ARGUS_OPT_SEGMENT_RASTER
    // argus_background_map / argus_detect_sources: cell grid, per-tile (base, count) + offsets, record staging
    struct BgScratch {
        float* cells; size_t cap_cells;          // med | sig | ngood, cap_cells each
        uint2* tiles; size_t cap_tiles;          // tile_info | offsets (4 B) behind it
        ArgusSourceRec* tmp; size_t cap_tmp;
        uint2* ord;                              // (band-local raster key, position in tmp) per record, cap_tmp entries
        unsigned* ctl;                           // [0] running total (atomics), [1] final count
        long long* h_n;                          // pinned
        unsigned char* cand; size_t cap_cand;    // argus_detect_frame: cuts, candidate lists, handed-over tiles (bytes)
        unsigned* last_fb;                       // device word: tiles the last argus_detect_frame scanned in full
    } bg;
    // argus_subtract_tiles: per-slice partial sums, per-tile fit, per-block (base, count) + offsets, record staging
    struct SubScratch {
        double* partial; float2* fit; size_t cap_tiles;
        uint2* blocks; size_t cap_blocks;           // block_info | offsets (4 B) behind it
        ArgusTransientRec* tmp; size_t cap_tmp;
        unsigned* ctl;                              // [0] running total (atomics), [1] final count
        long long* h_n;                             // pinned
    } sub;
};

static const double kPi = 3.14159265358979323846264338327950288;

#define CUDA_TRY(ctx, expr)                          \
    do {                                             \
        cudaError_t e_ = (expr);                     \
        if (e_ != cudaSuccess) {                     \
            if (ctx) (ctx)->last_cuda = (int)e_;     \
            return ARGUS_ERR_CUDA;                   \
        }                                            \
    } while (0)

extern "C" const char* argus_strerror(int s) {
    switch (s) {
        case ARGUS_OK: return "ok";
        case ARGUS_ERR_NULL: return "required pointer is NULL";
        case ARGUS_ERR_SHAPE: return "size argument out of range";
        case ARGUS_ERR_NSIDE: return "nside must be a power of two in [32, 2^29]";
        case ARGUS_ERR_KERNEL: return "unknown interpolation kernel";
        case ARGUS_ERR_WCS: return "invalid WCS (singular CD, non-finite value or bad sip_order)";
        case ARGUS_ERR_CAPACITY: return "capacity too small";
        case ARGUS_ERR_ALIGN: return "pointer not aligned to its element type";
        case ARGUS_ERR_CUDA: return "CUDA runtime error (see argus_last_cuda_error)";
        case ARGUS_ERR_STATE: return "call sequence error";
        default: return "unknown status";
    }
}

extern "C" int argus_version(void) { return ARGUS_VERSION_NUM; }

// ---------------------------------------------------------------------------------------- context
// Pseudo-inverse (A^T A)^-1 A^T of the design matrix of the 5x5 node grid S, T in {-1,-.5,0,.5,1} for the
// total-degree-`deg` basis U^i V^j ordered by degree, then by j: nc = (deg+1)(deg+2)/2 rows of 25.
static void lsq_pinv(int deg, double* pinv) {
    const int nc = (deg + 1) * (deg + 2) / 2;
    double A[25][15];
    for (int n = 0; n < 25; ++n) {
        double S = -1.0 + 0.5 * (n % 5), T = -1.0 + 0.5 * (n / 5);
        for (int d = 0; d <= deg; ++d)
            for (int j = 0; j <= d; ++j) A[n][d * (d + 1) / 2 + j] = pow(S, d - j) * pow(T, j);
    }
    double G[15][30];
    for (int i = 0; i < nc; ++i)
        for (int j = 0; j < nc; ++j) {
            double s = 0;
            for (int n = 0; n < 25; ++n) s += A[n][i] * A[n][j];
            G[i][j] = s;
            G[i][nc + j] = (i == j) ? 1.0 : 0.0;
        }
    for (int c = 0; c < nc; ++c) {   // Gauss-Jordan with partial pivoting
        int piv = c;
        for (int r = c + 1; r < nc; ++r)
            if (fabs(G[r][c]) > fabs(G[piv][c])) piv = r;
        if (piv != c)
            for (int j = 0; j < 2 * nc; ++j) { double t = G[c][j]; G[c][j] = G[piv][j]; G[piv][j] = t; }
        double d = 1.0 / G[c][c];
        for (int j = 0; j < 2 * nc; ++j) G[c][j] *= d;
        for (int r = 0; r < nc; ++r)
            if (r != c) {
                double fct = G[r][c];
                for (int j = 0; j < 2 * nc; ++j) G[r][j] -= fct * G[c][j];
            }
    }
    for (int i = 0; i < nc; ++i)
        for (int n = 0; n < 25; ++n) {
            double s = 0;
            for (int j = 0; j < nc; ++j) s += G[i][nc + j] * A[n][j];
            pinv[i * 25 + n] = s;
        }
}

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// One set of plan scratch: a single device allocation carved into the PlanBuffers arrays.
static cudaError_t alloc_plan_slot(int64_t max_tiles, int64_t max_slots, PlanBuffers& pb, void** block) {
    pb.max_tiles = (int)max_tiles;
    pb.max_slots = (int)max_slots;
    pb.max_hard = (int)(max_tiles / 4 < 1024 ? 1024 : max_tiles / 4);
    size_t o = 0, o_flag, o_bc, o_tid, o_rec, o_cnt, o_off, o_nt, o_hc, o_hl, o_mask, o_stats, o_pinv, o_dc, o_cls, o_bs, o_bb, o_fr, o_sc, o_sl, o_bid, o_nb, o_fc, o_fl, o_tk, o_p4, o_bc2, o_sp, o_cs;
    o_flag = o;  o = align_up(o + (size_t)pb.max_slots, 256);
    o_bc = o;    o = align_up(o + sizeof(int) * (pb.max_slots / 256 + 1), 256);
    o_tid = o;   o = align_up(o + sizeof(long long) * pb.max_tiles, 256);
    o_rec = o;   o = align_up(o + sizeof(TileRec) * pb.max_tiles, 256);
    o_cnt = o;   o = align_up(o + sizeof(int) * pb.max_tiles, 256);
    o_off = o;   o = align_up(o + sizeof(int) * (pb.max_tiles + 1), 256);
    o_cls = o;   o = align_up(o + (size_t)pb.max_tiles, 256);
    o_bs = o;    o = align_up(o + sizeof(int) * (pb.max_tiles / 1024 + 2), 256);
    o_bb = o;    o = align_up(o + sizeof(long long) * (pb.max_tiles / 1024 + 2), 256);
    o_nt = o;    o = align_up(o + sizeof(int), 256);
    o_hc = o;    o = align_up(o + sizeof(int), 256);
    o_hl = o;    o = align_up(o + sizeof(int) * pb.max_hard, 256);
    o_mask = o;  o = align_up(o + sizeof(unsigned) * 32 * (size_t)pb.max_hard, 256);
    o_stats = o; o = align_up(o + sizeof(PlanStats), 256);
    o_pinv = o;  o = align_up(o + sizeof(double) * 250, 256);
    o_dc = o;    o = align_up(o + sizeof(double) * 20 * (size_t)pb.max_tiles, 256);
    o_fr = o;    o = align_up(o + sizeof(FastRec) * (size_t)pb.max_tiles, 256);
    o_sc = o;    o = align_up(o + sizeof(int), 256);
    o_sl = o;    o = align_up(o + sizeof(int) * (size_t)pb.max_tiles, 256);   // any tile may end up on the slow list
    o_sp = o;    o = align_up(o + sizeof(int), 256);
    o_cs = o;    o = align_up(o + sizeof(long long) * (size_t)pb.max_tiles, 256);
    o_bid = o;   o = align_up(o + sizeof(long long) * (pb.max_tiles / 64 + 1), 256);
    o_nb = o;    o = align_up(o + sizeof(int), 256);
    o_fc = o;    o = align_up(o + sizeof(int), 256);
    o_fl = o;    o = align_up(o + sizeof(int) * (size_t)pb.max_tiles, 256);
    o_tk = o;    o = align_up(o + sizeof(unsigned), 256);
    o_p4 = o;    o = align_up(o + sizeof(double) * 375, 256);
    o_bc2 = o;   o = align_up(o + sizeof(double) * 32 * (size_t)(pb.max_tiles / 64 + 1), 256);
    cudaError_t e = cudaMalloc(block, o);
    if (e == cudaSuccess) e = cudaMemset(*block, 0, o);
    if (e != cudaSuccess) return e;
    char* b = (char*)*block;
    pb.slot_flag = (unsigned char*)(b + o_flag);
    pb.block_count = (int*)(b + o_bc);
    pb.tile_id = (long long*)(b + o_tid);
    pb.rec = (TileRec*)(b + o_rec);
    pb.tile_count = (int*)(b + o_cnt);
    pb.tile_offset = (int*)(b + o_off);
    pb.tile_cls = (unsigned char*)(b + o_cls);
    pb.block_sum = (int*)(b + o_bs);
    pb.block_base = (long long*)(b + o_bb);
    pb.n_tiles = (int*)(b + o_nt);
    pb.hard_count = (int*)(b + o_hc);
    pb.hard_list = (int*)(b + o_hl);
    pb.masks = (unsigned*)(b + o_mask);
    pb.stats = (PlanStats*)(b + o_stats);
    pb.pinv = (double*)(b + o_pinv);
    pb.dcoef = (double*)(b + o_dc);
    pb.frec = (FastRec*)(b + o_fr);
    pb.slow_count = (int*)(b + o_sc);
    pb.slow_list = (int*)(b + o_sl);
    pb.slow_plan = (int*)(b + o_sp);
    pb.cslot = (long long*)(b + o_cs);
    pb.block_id = (long long*)(b + o_bid);
    pb.n_blocks = (int*)(b + o_nb);
    pb.fb_count = (int*)(b + o_fc);
    pb.fb_list = (int*)(b + o_fl);
    pb.ticket = (unsigned*)(b + o_tk);
    pb.pinv4 = (double*)(b + o_p4);
    pb.bcoef = (double*)(b + o_bc2);
    double pinv[250], pinv4[375];
    lsq_pinv(3, pinv);
    lsq_pinv(4, pinv4);
    e = cudaMemcpy(pb.pinv, pinv, sizeof(pinv), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(pb.pinv4, pinv4, sizeof(pinv4), cudaMemcpyHostToDevice);
    return e;
}

// (Re)allocates the PLAN_SLOTS sets of plan scratch for max_tiles candidate tiles and max_slots scan slots.
static int alloc_plan_slots(argus_ctx* c, int64_t max_tiles, int64_t max_slots) {
    if (c->slot_block[0]) {
        CUDA_TRY(c, cudaDeviceSynchronize());        // plans and kernels still reading the old sets
        for (int sidx = 0; sidx < PLAN_SLOTS; ++sidx) { cudaFree(c->slot_block[sidx]); c->slot_block[sidx] = nullptr; c->slot_used[sidx] = false; }
    }
    c->plan_valid = false;
    c->cap_tiles = 0;
    for (int sidx = 0; sidx < PLAN_SLOTS; ++sidx) {
        CUDA_TRY(c, alloc_plan_slot(max_tiles, max_slots, c->slot_pb[sidx], &c->slot_block[sidx]));
        c->slot_pb[sidx].latch = c->d_latch;
    }
    c->pb = c->slot_pb[0];
    c->cur_slot = 0;
    c->cap_tiles = max_tiles;
    c->cap_slots = max_slots;
    return ARGUS_OK;
}

static int64_t default_max_slots(int64_t max_tiles) { return max_tiles * 8 < (1 << 26) ? max_tiles * 8 : (1 << 26); }

extern "C" int argus_ctx_create(argus_ctx** out, int device, int64_t max_tiles) {
    if (!out) return ARGUS_ERR_NULL;
    *out = nullptr;
    if (max_tiles != 0 && (max_tiles < 64 || max_tiles > (1 << 24))) return ARGUS_ERR_SHAPE;
    argus_ctx* c = new (std::nothrow) argus_ctx();
    if (!c) return ARGUS_ERR_CAPACITY;
    memset(c, 0, sizeof(*c));
    c->device = device;
    c->plan_cache = true;
    c->fast_enabled = true;
    c->unit_enabled = true;
    c->lz_small_enabled = true;
    c->auto_tiles = max_tiles == 0;
    cudaError_t e = cudaSetDevice(device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, device);
    if (e != cudaSuccess) { delete c; return ARGUS_ERR_CUDA; }
    cudaError_t e2 = cudaMalloc((void**)&c->d_latch, 4 * sizeof(int));     // + [2], [3]: the tile kernel's claim / finish counters
    if (e2 == cudaSuccess) e2 = cudaMemset(c->d_latch, 0, 4 * sizeof(int));
    if (e2 == cudaSuccess) e2 = cudaMallocHost((void**)&c->h_latch, 2 * sizeof(int));
    if (e2 == cudaSuccess) e2 = cudaMallocHost((void**)&c->h_stats, sizeof(PlanStats));
    int rc_slots = ARGUS_OK;
    if (e2 == cudaSuccess && !c->auto_tiles) rc_slots = alloc_plan_slots(c, max_tiles, default_max_slots(max_tiles));
    int prio_lo = 0, prio_hi = 0;
    if (e2 == cudaSuccess) e2 = cudaDeviceGetStreamPriorityRange(&prio_lo, &prio_hi);
    for (int i = 0; i < 2 && e2 == cudaSuccess; ++i) e2 = cudaStreamCreateWithPriority(&c->side[i], cudaStreamNonBlocking, prio_hi);
    for (int sidx = 0; sidx < PLAN_SLOTS && e2 == cudaSuccess; ++sidx) {
        e2 = cudaEventCreateWithFlags(&c->ev_done[sidx], cudaEventDisableTiming);
        if (e2 == cudaSuccess) e2 = cudaEventCreateWithFlags(&c->ev_free[sidx], cudaEventDisableTiming);
    }
    if (e2 != cudaSuccess || rc_slots != ARGUS_OK) {
        for (int sidx = 0; sidx < PLAN_SLOTS; ++sidx) if (c->slot_block[sidx]) cudaFree(c->slot_block[sidx]);
        if (c->h_stats) cudaFreeHost(c->h_stats);
        if (c->h_latch) cudaFreeHost(c->h_latch);
        if (c->d_latch) cudaFree(c->d_latch);
        delete c;
        return ARGUS_ERR_CUDA;
    }
    c->overlap = true;
    for (int i = 0; i < 256; ++i)
        for (int j = 0; j < 4; ++j) cudaEventCreate(&c->ev[i][j]);
    *out = c;
    return ARGUS_OK;
}

extern "C" int argus_ctx_destroy(argus_ctx* c) {
    if (!c) return ARGUS_ERR_NULL;
    cudaSetDevice(c->device);
    for (int i = 0; i < 2; ++i) cudaStreamSynchronize(c->side[i]);   // plans still running underneath the caller's kernels
    for (int i = 0; i < 256; ++i)
        for (int j = 0; j < 4; ++j) cudaEventDestroy(c->ev[i][j]);
    for (int sidx = 0; sidx < PLAN_SLOTS; ++sidx) {
        if (c->slot_block[sidx]) cudaFree(c->slot_block[sidx]);
        if (c->unit_block[sidx]) cudaFree(c->unit_block[sidx]);
        cudaEventDestroy(c->ev_done[sidx]);
        cudaEventDestroy(c->ev_free[sidx]);
    }
    for (int i = 0; i < 2; ++i) cudaStreamDestroy(c->side[i]);
    if (c->s_up) { cudaStreamSynchronize(c->s_up); cudaStreamDestroy(c->s_up); }
    if (c->s_down) { cudaStreamSynchronize(c->s_down); cudaStreamDestroy(c->s_down); }
    for (int i = 0; i < 2; ++i) {
        if (c->hb[i].raw) cudaFree(c->hb[i].raw);
        if (c->hb[i].val) cudaFree(c->hb[i].val);
        if (c->hb[i].wgt) cudaFree(c->hb[i].wgt);
        if (c->hb[i].idx) cudaFree(c->hb[i].idx);
        if (c->hb[i].seg16) cudaFree(c->hb[i].seg16);
        if (c->hb[i].mini_id) cudaFree(c->hb[i].mini_id);
        if (c->hb[i].mini_val) cudaFree(c->hb[i].mini_val);
        if (c->hb[i].mini_wgt) cudaFree(c->hb[i].mini_wgt);
        if (c->hb[i].n_mini) cudaFree(c->hb[i].n_mini);
        if (c->hb[i].ev_ok) { cudaEventDestroy(c->hb[i].up); cudaEventDestroy(c->hb[i].run); cudaEventDestroy(c->hb[i].down); }
    }
    if (c->seg.mini_start) cudaFree(c->seg.mini_start);
    if (c->seg.ctl) cudaFree(c->seg.ctl);
    if (c->seg.h_n) cudaFreeHost(c->seg.h_n);
    if (c->bg.cells) cudaFree(c->bg.cells);
    if (c->bg.cand) cudaFree(c->bg.cand);
    if (c->bg.tiles) cudaFree(c->bg.tiles);
    if (c->bg.tmp) cudaFree(c->bg.tmp);
    if (c->bg.ord) cudaFree(c->bg.ord);
    if (c->bg.ctl) cudaFree(c->bg.ctl);
    if (c->bg.h_n) cudaFreeHost(c->bg.h_n);
    if (c->sub.partial) cudaFree(c->sub.partial);
    if (c->sub.fit) cudaFree(c->sub.fit);
    if (c->sub.blocks) cudaFree(c->sub.blocks);
    if (c->sub.tmp) cudaFree(c->sub.tmp);
    if (c->sub.ctl) cudaFree(c->sub.ctl);
    if (c->sub.h_n) cudaFreeHost(c->sub.h_n);
    cudaFreeHost(c->h_stats);
    cudaFreeHost(c->h_latch);
    cudaFree(c->d_latch);
    delete c;
    return ARGUS_OK;
}

extern "C" int argus_ctx_set_option(argus_ctx* c, int option, int64_t value) {
    if (!c) return ARGUS_ERR_NULL;
    if (option == ARGUS_OPT_PLAN_CACHE) {
        c->plan_cache = value != 0;
        if (!c->plan_cache) c->plan_valid = false;
        return ARGUS_OK;
    }
    if (option == ARGUS_OPT_PROFILE) {
        c->profile = value != 0;
        c->prof_n = 0;
        return ARGUS_OK;
    }
    if (option == ARGUS_OPT_PLAN_OVERLAP) {
        c->overlap = value != 0;
        return ARGUS_OK;
    }
    if (option == ARGUS_OPT_SEGMENT_RASTER) {
        c->seg_raster = value != 0;
        return ARGUS_OK;
    }
    if (option == ARGUS_OPT_UNIT_MARGIN) {
        if (value < -8 || value > 40) return ARGUS_ERR_SHAPE;     // 9 .. 40: self-test of the ARGUS_DEBUG_BOUNDS check (box pretended value - 8 narrower)
        c->unit_margin = (int)value;
        c->plan_valid = false;
        return ARGUS_OK;
    }
    if (option == ARGUS_OPT_FAST_PATH) {
        c->fast_enabled = value != 0;
        c->unit_enabled = value == 1 || value == 3 || value == 4;
        c->unit_forced = value == 3;
        c->lz_small_enabled = value != 4;
        return ARGUS_OK;
    }
    return ARGUS_ERR_SHAPE;
}

extern "C" int argus_profile_read(argus_ctx* c, double* plan_ms, double* kernel_ms, int64_t* n_calls, void* stream) {
    if (!c || !plan_ms || !kernel_ms || !n_calls) return ARGUS_ERR_NULL;
    CUDA_TRY(c, cudaSetDevice(c->device));
    CUDA_TRY(c, cudaStreamSynchronize((cudaStream_t)stream));
    int n = c->prof_n < 256 ? c->prof_n : 256;
    double p = 0, k = 0;
    for (int i = 0; i < n; ++i) {
        float a = 0.f, b = 0.f;
        if (c->ev_plan[i]) CUDA_TRY(c, cudaEventElapsedTime(&a, c->ev[i][0], c->ev[i][1]));
        CUDA_TRY(c, cudaEventElapsedTime(&b, c->ev[i][2], c->ev[i][3]));
        p += a; k += b;
    }
    *plan_ms = p; *kernel_ms = k; *n_calls = n;
    c->prof_n = 0;
    return ARGUS_OK;
}

extern "C" int argus_last_cuda_error(const argus_ctx* c) { return c ? c->last_cuda : 0; }
extern "C" int64_t argus_launch_count(const argus_ctx* c) { return c ? c->n_launches : 0; }

// ------------------------------------------------------------------------------- frame constants
static bool is_pow2(int64_t v) { return v > 0 && (v & (v - 1)) == 0; }
static int ilog2(int64_t v) { int k = 0; while ((1ll << k) < v) ++k; return k; }

static int make_devwcs(const argus_wcs* w, int64_t W, int64_t H, int64_t nside, DevWcs* d, double* rho_max,
                       double* scale_rad) {
    if (W < 1 || H < 1 || W > (1 << 20) || H > (1 << 20)) return ARGUS_ERR_SHAPE;
    if (!is_pow2(nside) || nside < 32 || nside > (1ll << 29)) return ARGUS_ERR_NSIDE;
    if (w->sip_order < 0 || w->sip_order > 5 || w->sip_order == 1) return ARGUS_ERR_WCS;
    const double* v = &w->crval[0];
    for (int i = 0; i < 8; ++i)
        if (!isfinite(v[i])) return ARGUS_ERR_WCS;   // crval, crpix, cd are contiguous doubles
    for (int i = 0; i < 36; ++i)
        if (!isfinite(w->ap[i]) || !isfinite(w->bp[i])) return ARGUS_ERR_WCS;
    double det = w->cd[0][0] * w->cd[1][1] - w->cd[0][1] * w->cd[1][0];
    if (!(fabs(det) > 1e-300)) return ARGUS_ERR_WCS;
    double a0 = w->crval[0] * kPi / 180.0, d0 = w->crval[1] * kPi / 180.0;
    double sa = sin(a0), ca = cos(a0), sd = sin(d0), cd = cos(d0);
    d->er[0] = cd * ca; d->er[1] = cd * sa; d->er[2] = sd;
    d->ee[0] = -sa;     d->ee[1] = ca;      d->ee[2] = 0.0;
    d->en[0] = -sd * ca; d->en[1] = -sd * sa; d->en[2] = cd;
    double r2d = 180.0 / kPi;
    d->m[0][0] = w->cd[1][1] / det * r2d;  d->m[0][1] = -w->cd[0][1] / det * r2d;
    d->m[1][0] = -w->cd[1][0] / det * r2d; d->m[1][1] = w->cd[0][0] / det * r2d;
    d->crpix[0] = w->crpix[0]; d->crpix[1] = w->crpix[1];
    double s_rad = sqrt(fabs(det)) * kPi / 180.0;
    double rho = atan(1.25 * s_rad * hypot((double)W, (double)H) / 2.0);
    d->cos_rho = cos(rho);
    d->rho = rho;
    for (int i = 0; i < 36; ++i) { d->ap[i] = w->ap[i]; d->bp[i] = w->bp[i]; }
    d->sip_order = w->sip_order;
    d->W = (int)W; d->H = (int)H;
    d->k = ilog2(nside);
    d->nside = (double)nside;
    d->tile_ang = 1.3 * 32.0 / (double)nside;
    *rho_max = rho;
    *scale_rad = s_rad;
    return ARGUS_OK;
}

// host-side centre of a nested cell (only used to pick the coarse candidate cells)
static void host_cell_centre(int64_t nside, int64_t p, double v[3]) {
    int k = ilog2(nside), face, ix, iy;
    nest_to_xyf(p, k, face, ix, iy);
    double ns = (double)nside;
    int64_t jr = (int64_t)face_ring_offset(face) * nside - ix - iy - 1;
    double z, sth, nr;
    if (jr < nside) { nr = (double)jr; double t = nr * nr / (3 * ns * ns); z = 1 - t; sth = sqrt(t * (2 - t)); }
    else if (jr > 3 * nside) { nr = (double)(4 * nside - jr); double t = nr * nr / (3 * ns * ns); z = t - 1; sth = sqrt(t * (2 - t)); }
    else { nr = ns; z = (2.0 / 3.0) * (2.0 - jr / ns); sth = sqrt((1 - z) * (1 + z)); }
    double phi = (kPi / 4) * (face_phi_offset(face) + (double)(ix - iy) / nr);
    v[0] = sth * cos(phi); v[1] = sth * sin(phi); v[2] = z;
}

static void coarse_descend(const double er[3], double rho, int64_t nside_c, int64_t p, int64_t stop,
                           std::vector<long long>& out) {
    double v[3];
    host_cell_centre(nside_c, p, v);
    double dx = v[0] - er[0], dy = v[1] - er[1], dz = v[2] - er[2];
    double ang = 2.0 * asin(fmin(1.0, 0.5 * sqrt(dx * dx + dy * dy + dz * dz)));
    if (ang > rho + 1.3 / (double)nside_c) return;
    if (nside_c >= stop) { out.push_back(p); return; }
    for (int c = 0; c < 4; ++c) coarse_descend(er, rho, 2 * nside_c, 4 * p + c, stop, out);
}

static bool same_key(const argus_ctx* c, const argus_wcs* w, int64_t W, int64_t H, int64_t nside) {
    return c->plan_cache && c->plan_valid && c->key_W == W && c->key_H == H && c->key_nside == nside &&
           memcmp(&c->key_wcs, w, sizeof(argus_wcs)) == 0;
}

// Enqueue the plan kernels (A0 + A1).  No host synchronisation.
static int fast_stage_cap(const argus_ctx* c, int fast_kernel) {
    return fast_kernel == ARGUS_LANCZOS3 ? (c->lz_small ? FastCfg<1, 1>::CAP : FastCfg<1, 0>::CAP) : FastCfg<0, 0>::CAP;
}
static bool plan_usable(const argus_ctx* c, const argus_wcs* w, int64_t W, int64_t H, int64_t nside, bool need_full, int fast_kernel,
                        const UnitGeom* ug) {
    // the fast kernel's boxes are sized for one interpolation kernel's taps and one stage capacity; the general kernel does not care
    return same_key(c, w, W, H, nside) && (!need_full || c->plan_full) &&
           (fast_kernel < 0 || (c->plan_fast_kernel == (fast_kernel == ARGUS_LANCZOS3 ? 1 : 0) && (ug || c->plan_fast_cap == fast_stage_cap(c, fast_kernel)))) &&
           (ug ? (c->plan_unit && memcmp(&c->plan_geom, ug, sizeof(UnitGeom)) == 0) : (fast_kernel < 0 || !c->plan_unit));
}

// fast_kernel: interpolation kernel the fast (TMA-staged) kernel will run with, -1 = general kernel only (full plan).
// Scratch of the image-aligned units (resample_unit.cuh), one set per plan slot: segment counts (+ the stray counter),
// segment records, stray list.  Grown on demand (synchronises the device).
static int ensure_unit_scratch(argus_ctx* c, size_t n_units, int max_stray) {
    if (c->unit_block[0] && c->unit_cap >= n_units) return ARGUS_OK;
    if (c->unit_block[0]) {
        CUDA_TRY(c, cudaDeviceSynchronize());
        for (int sidx = 0; sidx < PLAN_SLOTS; ++sidx) { cudaFree(c->unit_block[sidx]); c->unit_block[sidx] = nullptr; }
    }
    c->plan_valid = false;
    const size_t want = align_up(n_units + 1, 1024);
    const size_t o_seg = align_up((want + 2) * sizeof(int), 256), o_stray = o_seg + align_up(want * UNIT_MAXSEG * sizeof(UnitSeg), 256);
    const size_t total = o_stray + 2 * (size_t)max_stray * sizeof(int);
    for (int sidx = 0; sidx < PLAN_SLOTS; ++sidx) {
        CUDA_TRY(c, cudaMalloc(&c->unit_block[sidx], total));
        char* b = (char*)c->unit_block[sidx];
        c->slot_ub[sidx].nseg = (int*)b;
        c->slot_ub[sidx].stray_count = (int*)b + n_units;      // zeroed together with nseg; re-pointed below when n_units changes
        c->slot_ub[sidx].seg = (UnitSeg*)(b + o_seg);
        c->slot_ub[sidx].stray_list = (int*)(b + o_stray);
    }
    c->unit_cap = want - 1;
    return ARGUS_OK;
}

// ug: unit geometry when the image-aligned unit kernel will run the frame (segment lists are built), else NULL.
static int build_plan(argus_ctx* c, const argus_wcs* w, int64_t W, int64_t H, int64_t nside, long long out_cap,
                      cudaStream_t caller, int fast_kernel, int prof_slot, const UnitGeom* ug = nullptr) {
    // Lanczos-3: any tile may be handed to the general kernel at run time (masked pixels in its box) => full records
    const bool need_full = fast_kernel != ARGUS_BILINEAR && !ug;      // (the unit kernel hands over to the stray kernel instead)
    DevWcs dw;
    double rho, s_rad;
    int rc = make_devwcs(w, W, H, nside, &dw, &rho, &s_rad);
    if (rc) return rc;
    if (plan_usable(c, w, W, H, nside, need_full, fast_kernel, ug)) {
        if (out_cap >= 0) {   // cached plan: the capacity of THIS call's outputs still has to be checked
            plan_check_capacity_kernel<<<1, 32, 0, caller>>>(c->pb, out_cap);
            c->n_launches++;
        }
        return ARGUS_OK;
    }
    c->plan_valid = false;
    const int lite = need_full ? 0 : 1;
    // Hierarchical plan (plan_block.cuh) whenever a block of 8x8 tiles exists at this nside; the flat plan (one
    // scan slot and one fit per tile) serves nside < 256.
    const bool blocks = dw.k >= ARGUS_TILE_LOG2 + BLOCK_TILES_LOG2;
    int64_t nside_t = nside >> ARGUS_TILE_LOG2;                      // tile-level nside
    if (nside_t < 1) nside_t = 1;
    int64_t nside_s = blocks ? (nside_t >> BLOCK_TILES_LOG2) : nside_t;   // resolution of the scan slots
    // coarse resolution: cells comparable to the search cone, list passed by value
    int64_t nside_c = 1;
    while (nside_c < nside_s && (double)nside_c < 2.0 / rho) nside_c <<= 1;
    std::vector<long long> cells;
    for (;;) {
        cells.clear();
        for (int b = 0; b < 12; ++b) coarse_descend(dw.er, rho, 1, b, nside_c, cells);
        if ((int)cells.size() <= ARGUS_MAX_COARSE || nside_c == 1) break;
        nside_c >>= 1;
    }
    if ((int)cells.size() > ARGUS_MAX_COARSE) return ARGUS_ERR_CAPACITY;
    CoarseList cl;
    memset(&cl, 0, sizeof(cl));
    cl.n = (int)cells.size();
    cl.ratio_log2 = ilog2(nside_s / nside_c);
    for (int i = 0; i < cl.n; ++i) cl.cell[i] = cells[i];
    long long n_slots = (long long)cl.n << (2 * cl.ratio_log2);
    if (cl.ratio_log2 > 12) return ARGUS_ERR_CAPACITY;
    if (c->auto_tiles) {
        // Scratch sized for this frame: candidate tiles = tiles whose block centre lies within one block radius of the
        // frame, i.e. (W + 2 r)(H + 2 r) detector pixels' worth of HEALPix pixels (equal area), + 50 % and a margin for
        // the ragged block boundary; never more than the scan's own bound.  Grown (device synchronised) when a larger
        // frame arrives, never shrunk.
        const double omega = 4.0 * kPi / (12.0 * (double)nside * (double)nside);
        const double unit_ang = (blocks ? 8.0 : 1.0) * dw.tile_ang;
        const double r_px = 1.05 * unit_ang / s_rad + 2.0;
        const double hp_px = ((double)W + 2.0 * r_px) * ((double)H + 2.0 * r_px) * s_rad * s_rad / omega;
        long long est = (long long)(1.5 * hp_px / 1024.0) + 4096;
        const long long bound = blocks ? n_slots * 64 : n_slots;
        if (est > bound) est = bound;
        if (est < 1024) est = 1024;
        est = (est + 1023) / 1024 * 1024;
        if (est > (1 << 24)) return ARGUS_ERR_CAPACITY;
        long long want_slots = n_slots > default_max_slots(est) ? n_slots : default_max_slots(est);
        if (want_slots > (1 << 26)) return ARGUS_ERR_CAPACITY;
        if (est > c->cap_tiles || want_slots > c->cap_slots) {
            int rc2 = alloc_plan_slots(c, est > c->cap_tiles ? est : c->cap_tiles, want_slots > c->cap_slots ? want_slots : c->cap_slots);
            if (rc2) return rc2;
        }
    }
    if (n_slots > c->slot_pb[0].max_slots) return ARGUS_ERR_CAPACITY;
    // where the plan is built: in place on the caller's stream, or (overlap) in the other scratch set on the side
    // stream, after the last kernel that read that set
    int ps = c->cur_slot;
    cudaStream_t st = caller;
    if (c->overlap) {
        ps = (c->cur_slot + 1) % PLAN_SLOTS;
        st = c->side[c->side_next];
        c->side_next ^= 1;
        if (c->slot_used[ps]) CUDA_TRY(c, cudaStreamWaitEvent(st, c->ev_free[ps], 0));
    }
    if (ug) {
        int rcu = ensure_unit_scratch(c, (size_t)ug->nux * (size_t)ug->nuy, ug->max_stray);
        if (rcu) return rcu;
    }
    c->pb = c->slot_pb[ps];
    c->pb.unit_mode = ug ? 1 : 0;
    c->cur_slot = ps;
    {   // tap apron and stage capacity the fast kernel's boxes are sized for (a full plan keeps bilinear boxes)
        const int fk = fast_kernel == ARGUS_LANCZOS3 ? 1 : 0;
        c->pb.fast_tl = fk ? FastCfg<1>::TL : FastCfg<0>::TL;
        c->pb.fast_tr = fk ? FastCfg<1>::TR : FastCfg<0>::TR;
        c->pb.fast_cap = fast_stage_cap(c, fast_kernel);
    }
    if (prof_slot >= 0) cudaEventRecord(c->ev[prof_slot][0], st);
    if (n_slots == 0) n_slots = 1;
    int nblk = (int)((n_slots + 255) / 256);
    long long tile_bound;
    if (blocks) {
        double block_ang = 8.0 * dw.tile_ang;
        double rad_px = 1.05 * block_ang / s_rad + 2.0;
        plan_bscan_kernel<<<nblk, 256, 0, st>>>(dw, cl, c->pb, rad_px, block_ang);
        int nb_bound = (int)(n_slots < c->pb.max_tiles / 64 ? n_slots : c->pb.max_tiles / 64);
        int g = (nb_bound + BFIT_WARPS - 1) / BFIT_WARPS;
        if (g > c->sm_count * 8) g = c->sm_count * 8;
        plan_blockfit_kernel<<<g < 1 ? 1 : g, 32 * BFIT_WARPS, 0, st>>>(dw, c->pb);
        int g2 = (nb_bound + 1) / 2;
        if (g2 > c->sm_count * 16) g2 = c->sm_count * 16;
        plan_tilegen_kernel<<<g2 < 1 ? 1 : g2, 128, 0, st>>>(dw, c->pb, lite);
        plan_fit_kernel<<<c->sm_count * 2, 32 * FIT_WARPS, 0, st>>>(dw, c->pb, 1, lite);
        tile_bound = n_slots * 64;
        c->n_launches += 4;
    } else {
        double rad_px = 1.05 * dw.tile_ang / s_rad + 2.0;
        plan_scan_kernel<<<nblk, 256, 0, st>>>(dw, cl, c->pb, rad_px);
        plan_compact_kernel<<<nblk, 256, 0, st>>>(cl, c->pb);
        plan_fit_kernel<<<c->sm_count * 4, 32 * FIT_WARPS, 0, st>>>(dw, c->pb, 0, lite);
        tile_bound = n_slots;
        c->n_launches += 3;
    }
    plan_members_kernel<<<c->sm_count * 16, 256, 0, st>>>(dw, c->pb);
    {
        long long bound = tile_bound < c->pb.max_tiles ? tile_bound : c->pb.max_tiles;
        int gb = (int)((bound + 1023) / 1024);
        plan_offsets_kernel<<<gb < 1 ? 1 : gb, 256, 0, st>>>(c->pb, out_cap);
    }
    c->n_launches += 2;
    if (ug) {   // segment lists of the image-aligned units (resample_unit.cuh)
        const size_t n_units = (size_t)ug->nux * (size_t)ug->nuy;
        c->slot_ub[ps].stray_count = c->slot_ub[ps].nseg + n_units;
        c->slot_ub[ps].stray_rt = c->slot_ub[ps].nseg + n_units + 1;
        CUDA_TRY(c, cudaMemsetAsync(c->slot_ub[ps].nseg, 0, (n_units + 2) * sizeof(int), st));
        {   // one warp per tile, all tiles in flight at once (the kernel is a chain of latencies per tile)
            long long bound = tile_bound < c->pb.max_tiles ? tile_bound : c->pb.max_tiles;
            int gu = (int)((bound + 7) / 8);
            plan_units_kernel<<<gu < 1 ? 1 : gu, 256, 0, st>>>(c->pb, *ug, c->slot_ub[ps]);
        }
        c->n_launches++;
    }
    CUDA_TRY(c, cudaGetLastError());
    if (prof_slot >= 0) cudaEventRecord(c->ev[prof_slot][1], st);
    if (c->overlap) {
        CUDA_TRY(c, cudaEventRecord(c->ev_done[ps], st));
        CUDA_TRY(c, cudaStreamWaitEvent(caller, c->ev_done[ps], 0));
    }
    c->dw = dw;
    c->key_wcs = *w;
    c->key_W = W; c->key_H = H; c->key_nside = nside;
    c->plan_valid = true;
    c->plan_full = need_full;
    c->plan_fast_kernel = fast_kernel == ARGUS_LANCZOS3 ? 1 : 0;
    c->plan_fast_cap = fast_stage_cap(c, fast_kernel);
    c->plan_unit = ug != nullptr;
    if (ug) c->plan_geom = *ug;
    return ARGUS_OK;
}

static bool aligned(const void* p, size_t a) { return ((uintptr_t)p % a) == 0; }

// The kernels just enqueued on `caller` read the current scratch set: a later plan into that set waits for them.
static void mark_slot_read(argus_ctx* c, cudaStream_t caller) {
    if (cudaEventRecord(c->ev_free[c->cur_slot], caller) == cudaSuccess) c->slot_used[c->cur_slot] = true;
}

static int make_frameargs(const argus_frame* fr, int64_t W, int64_t H, FrameArgs* f, bool* fused) {
    memset(f, 0, sizeof(*f));
    if (fr->raw && fr->masters_format != 0) {
        if (fr->masters_format != ARGUS_MASTERS_F32 && fr->masters_format != ARGUS_MASTERS_F16) return ARGUS_ERR_SHAPE;
        if (!fr->offset || !fr->gain) return ARGUS_ERR_NULL;
        if (fr->sat_adu < 0) return ARGUS_ERR_SHAPE;
        const size_t es = fr->masters_format == ARGUS_MASTERS_F32 ? 4 : 2;
        if (!aligned(fr->raw, 2) || !aligned(fr->offset, es) || !aligned(fr->gain, es)) return ARGUS_ERR_ALIGN;
        f->raw = fr->raw; f->offset = fr->offset; f->gain = fr->gain; f->pre = fr->masters_format;
        f->sat_adu = fr->sat_adu; f->t_exp = 0.f; f->flat_min = 1.f;
        f->vec_ok = (W % 4 == 0) && (W * H < (1ll << 31)) && aligned(fr->raw, 8) && aligned(fr->offset, 4 * es) && aligned(fr->gain, 4 * es);
        *fused = true;
    } else if (fr->raw) {
        if (!fr->bias || !fr->dark || !fr->flat) return ARGUS_ERR_NULL;
        if (!(fr->flat_min > 0.0f) || !(fr->flat_min < INFINITY) || fr->sat_adu < 0) return ARGUS_ERR_SHAPE;
        if (!aligned(fr->raw, 2) || !aligned(fr->bias, 4) || !aligned(fr->dark, 4) || !aligned(fr->flat, 4)) return ARGUS_ERR_ALIGN;
        f->raw = fr->raw; f->bias = fr->bias; f->dark = fr->dark; f->flat = fr->flat; f->bpm = fr->bpm;
        f->t_exp = fr->t_exp; f->flat_min = fr->flat_min; f->sat_adu = fr->sat_adu;
        f->vec_ok = (W % 4 == 0) && (W * H < (1ll << 31)) && aligned(fr->raw, 8) && aligned(fr->bias, 16) && aligned(fr->dark, 16) &&
                    aligned(fr->flat, 16) && (!fr->bpm || aligned(fr->bpm, 4));
        *fused = true;
    } else {
        if (!fr->cal || !fr->mask) return ARGUS_ERR_NULL;
        if (!aligned(fr->cal, 4)) return ARGUS_ERR_ALIGN;
        f->cal = fr->cal; f->mask = fr->mask;
        f->vec_ok = (W % 4 == 0) && (W * H < (1ll << 31)) && aligned(fr->cal, 16) && aligned(fr->mask, 4);
        *fused = false;
    }
    return ARGUS_OK;
}

// ------------------------------------------------------------------------------------- A2 standalone
extern "C" int argus_calibrate(argus_ctx* c, const uint16_t* raw, const float* bias, const float* dark,
                               const float* flat, const uint8_t* bpm, int64_t W, int64_t H, float t_exp,
                               int32_t sat_adu, float flat_min, float* cal_out, uint8_t* mask_out, void* stream) {
    if (!c || !raw || !bias || !dark || !flat || !cal_out || !mask_out) return ARGUS_ERR_NULL;
    if (W < 1 || H < 1 || W > (1 << 20) || H > (1 << 20)) return ARGUS_ERR_SHAPE;
    argus_frame fr;
    memset(&fr, 0, sizeof(fr));
    fr.raw = raw; fr.bias = bias; fr.dark = dark; fr.flat = flat; fr.bpm = bpm;
    fr.t_exp = t_exp; fr.sat_adu = sat_adu; fr.flat_min = flat_min;
    FrameArgs f;
    bool fused;
    int rc = make_frameargs(&fr, W, H, &f, &fused);
    if (rc) return rc;
    if (!aligned(cal_out, 4)) return ARGUS_ERR_ALIGN;
    long long n = W * H;
    // the flat vector path needs n % 4 == 0 and aligned outputs (rows need not be aligned: 1-D sweep)
    f.vec_ok = (n % 4 == 0) && aligned(raw, 8) && aligned(bias, 16) && aligned(dark, 16) && aligned(flat, 16) &&
               (!bpm || aligned(bpm, 4)) && aligned(cal_out, 16) && aligned(mask_out, 4);
    CUDA_TRY(c, cudaSetDevice(c->device));
    calibrate_kernel<<<c->sm_count * 8, 256, 0, (cudaStream_t)stream>>>(f, n, cal_out, mask_out);
    c->n_launches++;
    CUDA_TRY(c, cudaGetLastError());
    return ARGUS_OK;
}

// ------------------------------------------------------------------------ pre-fused masters (8(f).4)
extern "C" int argus_prepare_masters(argus_ctx* c, const float* bias, const float* dark, const float* flat, const uint8_t* bpm,
                                     int64_t W, int64_t H, float t_exp, float flat_min, int format, void* offset_out,
                                     void* gain_out, void* stream) {
    if (!c || !bias || !dark || !flat || !offset_out || !gain_out) return ARGUS_ERR_NULL;
    if (W < 1 || H < 1 || W > (1 << 20) || H > (1 << 20)) return ARGUS_ERR_SHAPE;
    if (format != ARGUS_MASTERS_F32 && format != ARGUS_MASTERS_F16) return ARGUS_ERR_SHAPE;
    if (!(flat_min > 0.0f) || !(flat_min < INFINITY) || !(fabsf(t_exp) < INFINITY)) return ARGUS_ERR_SHAPE;
    const size_t es = format == ARGUS_MASTERS_F32 ? 4 : 2;
    if (!aligned(bias, 4) || !aligned(dark, 4) || !aligned(flat, 4) || !aligned(offset_out, es) || !aligned(gain_out, es)) return ARGUS_ERR_ALIGN;
    CUDA_TRY(c, cudaSetDevice(c->device));
    const long long n = W * H;
    if (format == ARGUS_MASTERS_F32)
        prepare_masters_kernel<1><<<c->sm_count * 8, 256, 0, (cudaStream_t)stream>>>(bias, dark, flat, bpm, n, t_exp, flat_min, offset_out, gain_out);
    else
        prepare_masters_kernel<2><<<c->sm_count * 8, 256, 0, (cudaStream_t)stream>>>(bias, dark, flat, bpm, n, t_exp, flat_min, offset_out, gain_out);
    c->n_launches++;
    CUDA_TRY(c, cudaGetLastError());
    return ARGUS_OK;
}

// --------------------------------------------------------------------------------------- A0 + A1
// Plan statistics of the current scratch set + the context-wide overflow latch (read and cleared).
static int fetch_stats(argus_ctx* c, cudaStream_t st, int* latched) {
    *latched = 0;
    if (!c->slot_block[0]) { memset(c->h_stats, 0, sizeof(PlanStats)); return ARGUS_OK; }   // no plan built yet
    CUDA_TRY(c, cudaMemcpyAsync(c->h_stats, c->pb.stats, sizeof(PlanStats), cudaMemcpyDeviceToHost, st));
    plan_latch_fetch_kernel<<<1, 32, 0, st>>>(c->d_latch, c->d_latch + 1);
    c->n_launches++;
    CUDA_TRY(c, cudaMemcpyAsync(c->h_latch, c->d_latch + 1, sizeof(int), cudaMemcpyDeviceToHost, st));
    c->h_latch[1] = 0;
    if (c->plan_valid && c->plan_unit)
        CUDA_TRY(c, cudaMemcpyAsync(c->h_latch + 1, c->slot_ub[c->cur_slot].stray_count, sizeof(int), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(c, cudaStreamSynchronize(st));
    *latched = *c->h_latch;
    return ARGUS_OK;
}

extern "C" int argus_healpix_footprint(argus_ctx* c, const argus_wcs* wcs, int64_t W, int64_t H, int64_t nside,
                                       int64_t* idx_out, size_t capacity, size_t* n_out, void* stream) {
    if (!c || !wcs || !n_out) return ARGUS_ERR_NULL;
    if (idx_out && !aligned(idx_out, 8)) return ARGUS_ERR_ALIGN;
    cudaStream_t st = (cudaStream_t)stream;
    CUDA_TRY(c, cudaSetDevice(c->device));
    int rc = build_plan(c, wcs, W, H, nside, -1, st, -1, -1);
    if (rc) return rc;
    int latched;
    rc = fetch_stats(c, st, &latched);
    if (rc) return rc;
    *n_out = (size_t)c->h_stats->n_footprint;
    if (c->h_stats->overflow & 3) { c->plan_valid = false; return ARGUS_ERR_CAPACITY; }
    if (latched) return ARGUS_ERR_CAPACITY;      // an earlier asynchronous call overflowed (this plan itself is intact)
    if (idx_out) {
        if ((size_t)c->h_stats->n_footprint > capacity) return ARGUS_ERR_CAPACITY;
        plan_write_indices_kernel<<<c->sm_count * 8, 256, 0, st>>>(c->pb, (long long*)idx_out, (long long)capacity);
        c->n_launches++;
        CUDA_TRY(c, cudaGetLastError());
        CUDA_TRY(c, cudaStreamSynchronize(st));
    }
    return ARGUS_OK;
}

extern "C" int argus_plan_info(argus_ctx* c, argus_plan_stats* out, void* stream) {
    if (!c || !out) return ARGUS_ERR_NULL;
    CUDA_TRY(c, cudaSetDevice(c->device));
    int latched;
    int rc = fetch_stats(c, (cudaStream_t)stream, &latched);
    if (rc) return rc;
    const PlanStats* s = c->h_stats;
    out->n_footprint = s->n_footprint; out->n_tiles = s->n_tiles; out->n_inside = s->n_inside;
    out->n_border = s->n_border; out->n_exact = s->n_exact; out->n_empty = s->n_empty;
    out->n_units = (c->plan_valid && c->plan_unit) ? (int64_t)c->plan_geom.nux * c->plan_geom.nuy : 0;
    out->n_stray = c->h_latch[1];
    if (s->overflow) c->plan_valid = false;
    if (s->overflow || latched) return ARGUS_ERR_CAPACITY;
    return ARGUS_OK;
}

// ------------------------------------------------------------------------------------- A3..A6
// cuTensorMapEncodeTiled through the runtime's driver entry point (libargus.so has no link-time libcuda dependency,
// so it loads on a machine without a driver).
typedef CUresult (*encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                    const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// TMA descriptors for (raw, bias, dark, flat): 2-D tensors {W, H}, boxes {40..72 step 8} x {48, 56, 64, 72}, zero fill outside.
static bool fast_maps(argus_ctx* c, const FrameArgs& f, int64_t W, int64_t H) {
    if (!c->fast_enabled || !f.raw || f.bpm || f.pre) return false;
    if (W % 8 != 0 || W < 8 || !aligned(f.raw, 16) || !aligned(f.bias, 16) || !aligned(f.dark, 16) || !aligned(f.flat, 16)) return false;
    if (!c->encode_tried) {
        c->encode_tried = true;
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) == cudaSuccess &&
            qr == cudaDriverEntryPointSuccess)
            c->encode_fn = fn;
        else
            (void)cudaGetLastError();
    }
    if (!c->encode_fn) return false;
    const void* key[4] = {f.raw, f.bias, f.dark, f.flat};
    if (memcmp(key, c->maps_key, sizeof(key)) == 0 && c->maps_W == W && c->maps_H == H) return true;
    encode_tiled_fn enc = (encode_tiled_fn)c->encode_fn;
    for (int hc = 0; hc < 4; ++hc)
      for (int wc = 0; wc < 5; ++wc)
        for (int a = 0; a < 4; ++a) {
            cuuint64_t dims[2] = {(cuuint64_t)W, (cuuint64_t)H};
            cuuint64_t strides[1] = {(cuuint64_t)W * (a == 0 ? 2u : 4u)};
            cuuint32_t box[2] = {(cuuint32_t)(40 + 8 * wc), (cuuint32_t)(48 + 8 * hc)};
            cuuint32_t es[2] = {1, 1};
            CUresult r = enc(&c->maps.m[hc][wc][a], a == 0 ? CU_TENSOR_MAP_DATA_TYPE_UINT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2,
                             const_cast<void*>(key[a]), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                             CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
            if (r != CUDA_SUCCESS) { c->maps_W = -1; return false; }
        }
    memcpy(c->maps_key, key, sizeof(key));
    c->maps_W = W; c->maps_H = H;
    return true;
}

// ------------------------------------------------------------------------- image-aligned units: host side
static unsigned long long host_spread(unsigned v) {      // bit i -> bit 2 i
    unsigned long long r = 0;
    for (int b = 0; b < 32; ++b) r |= (unsigned long long)((v >> b) & 1u) << (2 * b);
    return r;
}

static void host_vec_to_xy(const DevWcs& w, const double v[3], double& x, double& y) {   // inverse TAN (+ SIP), as vec_to_xy
    const double cosc = v[0] * w.er[0] + v[1] * w.er[1] + v[2] * w.er[2], inv = 1.0 / cosc;
    const double xi = (v[0] * w.ee[0] + v[1] * w.ee[1] + v[2] * w.ee[2]) * inv, eta = (v[0] * w.en[0] + v[1] * w.en[1] + v[2] * w.en[2]) * inv;
    const double U = w.m[0][0] * xi + w.m[0][1] * eta, V = w.m[1][0] * xi + w.m[1][1] * eta;
    double fu = 0.0, fv = 0.0, up = 1.0;
    for (int p = 0; p <= w.sip_order && w.sip_order > 0; ++p) {
        double m = up;
        for (int q = 0; p + q <= w.sip_order; ++q) { fu += w.ap[p * 6 + q] * m; fv += w.bp[p * 6 + q] * m; m *= V; }
        up *= U;
    }
    x = U + fu + w.crpix[0];
    y = V + fv + w.crpix[1];
}

// Extent (cells) of a 4 x 4-pixel sub-block about its centre, per image axis: 1.5 (|dx/dix| + |dx/diy|) from the Jacobian
// of the pixel -> image mapping at the HEALPix pixel nearest to the sky direction v (descent by closest child centre).
static void unit_extent_at(const DevWcs& w, const argus_wcs* wc, int64_t nside, const double v[3], double& ex, double& ey) {
    long long p = 0;
    double best = -2.0;
    for (int b = 0; b < 12; ++b) {
        double c[3];
        host_cell_centre(1, b, c);
        const double d = c[0] * v[0] + c[1] * v[1] + c[2] * v[2];
        if (d > best) { best = d; p = b; }
    }
    for (int64_t ns = 2; ns <= nside; ns <<= 1) {
        long long bp = 4 * p;
        best = -2.0;
        for (int ch = 0; ch < 4; ++ch) {
            double c[3];
            host_cell_centre(ns, 4 * p + ch, c);
            const double d = c[0] * v[0] + c[1] * v[1] + c[2] * v[2];
            if (d > best) { best = d; bp = 4 * p + ch; }
        }
        p = bp;
    }
    const int k = ilog2(nside);
    int face, ix, iy;
    nest_to_xyf(p, k, face, ix, iy);
    const int dx = ix + 1 < nside ? 1 : -1, dy = iy + 1 < nside ? 1 : -1;
    double c0[3], c1[3], c2[3], x0, y0, x1, y1, x2, y2;
    const long long fb = (long long)face << (2 * k);
    host_cell_centre(nside, p, c0);
    host_cell_centre(nside, fb | (long long)(host_spread((unsigned)(ix + dx)) | (host_spread((unsigned)iy) << 1)), c1);
    host_cell_centre(nside, fb | (long long)(host_spread((unsigned)ix) | (host_spread((unsigned)(iy + dy)) << 1)), c2);
    host_vec_to_xy(w, c0, x0, y0); host_vec_to_xy(w, c1, x1, y1); host_vec_to_xy(w, c2, x2, y2);
    (void)wc;
    ex = 1.5 * (fabs(x1 - x0) + fabs(x2 - x0));
    ey = 1.5 * (fabs(y1 - y0) + fabs(y2 - y0));
}

// Unit geometry for (wcs, W, H, nside, kernel): false when units do not fit a stage (very coarse HEALPix pixels) -- the tile
// kernel or the general kernel then runs the frame.  The extents are ESTIMATES from nine sky directions (centre, corners,
// edge midpoints); a sub-block that exceeds them anyway is found by plan_units_kernel and served by the stray kernel.
static bool unit_geometry(const DevWcs& dw, const argus_wcs* w, int64_t W, int64_t H, int64_t nside, double s_rad, int kernel, UnitGeom* g,
                          bool* tiles_fit, bool* tiles_small, int margin_delta) {
    const int ktl = kernel == ARGUS_LANCZOS3 ? 2 : 0, ktr = kernel == ARGUS_LANCZOS3 ? 3 : 1;
    const int kcap = kernel == ARGUS_LANCZOS3 ? FAST_CAP_PX_LZ : FAST_CAP_PX;
    double ex = 0.0, ey = 0.0;
    *tiles_fit = true;
    *tiles_small = false;
    bool small = kernel == ARGUS_LANCZOS3;
    for (int sy = -1; sy <= 1; ++sy)
        for (int sx = -1; sx <= 1; ++sx) {
            const double px = 0.45 * sx * (double)W, py = 0.45 * sy * (double)H;       // pixel offsets from CRPIX (about the frame centre)
            const double d2r = kPi / 180.0;
            const double xi = (w->cd[0][0] * px + w->cd[0][1] * py) * d2r, eta = (w->cd[1][0] * px + w->cd[1][1] * py) * d2r;
            double v[3];
            for (int i = 0; i < 3; ++i) v[i] = dw.er[i] + xi * dw.ee[i] + eta * dw.en[i];
            const double nrm = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
            for (int i = 0; i < 3; ++i) v[i] /= nrm;
            double ax, ay;
            unit_extent_at(dw, w, nside, v, ax, ay);
            if (!(ax < 64.0) || !(ay < 64.0)) return false;
            ex = fmax(ex, ax); ey = fmax(ey, ay);
            {   // would a whole 32 x 32-pixel tile fit the tile kernel's stage here?  (mirror of fast_box, worst-case alignment)
                const int span_x = (int)ceil(31.0 / 1.5 * ax) + 3, span_y = (int)ceil(31.0 / 1.5 * ay) + 3;   // + tile-to-tile variation
                const int bw = span_x + ktl + ktr + 7, bh = span_y + ktl + ktr;
                const int boxw = bw <= 40 ? 40 : (bw + 7) / 8 * 8, boxh = bh <= 48 ? 48 : (bh + 7) / 8 * 8;
                if (bw > 72 || bh > 72 || boxw * boxh > kcap) *tiles_fit = false;
                if (boxw * boxh > FAST_CAP_PX_LZ_SMALL || bh * fast_cal_pitch(boxw) > FAST_CAP_PX_LZ_SMALL * 9 / 8) small = false;
            }
        }
    *tiles_small = small && *tiles_fit;
    memset(g, 0, sizeof(*g));
    g->tl = ktl; g->tr = ktr;
    const int chk = margin_delta > 8 ? margin_delta - 8 : 0;
    if (margin_delta > 8) margin_delta = 0;
    g->Mx = (int)ceil(1.03 * ex + 0.02) + margin_delta; g->My = (int)ceil(1.03 * ey + 0.02) + margin_delta;
    if (g->Mx < 0) g->Mx = 0;
    if (g->My < 0) g->My = 0;
    g->BW = UNIT_BOXW;
    g->RW = (g->BW - 2 * g->Mx - g->tl - g->tr) & ~7;
    int bh = UNIT_CAP / g->BW;
    g->RH = bh - 2 * g->My - g->tl - g->tr;
    if (g->RW < 16 || g->RH < 8) return false;
    // sub-blocks per unit: owned cells x HEALPix pixels per cell / 16; keep the expected number below 0.55 of the list
    const double hp_per_cell = s_rad * s_rad / (4.0 * kPi / (12.0 * (double)nside * (double)nside));
    while (g->RH > 8 && (double)g->RW * g->RH * hp_per_cell / 16.0 > 0.55 * UNIT_MAXSB) g->RH -= 2;
    if ((double)g->RW * g->RH * hp_per_cell / 16.0 > 0.55 * UNIT_MAXSB) return false;
    if ((double)g->RW * g->RH * hp_per_cell < 64.0) return false;     // a handful of outputs per unit: not worth a stage
    g->BH = g->RH + 2 * g->My + g->tl + g->tr;
    // the centre of a border tile's sub-block can lie up to its extent outside the frame: the grid starts at or below cell
    // -(M + 2) and ends at or beyond cell W + M + 1
    const int kx = (2 * g->Mx + g->tl + 2 + 7) / 8;
    g->x_off = g->Mx + g->tl - 8 * kx;                                  // <= -(Mx + 2) and (x_off - Mx - tl) % 8 == 0
    g->y_off = -(g->My + 2);
    g->nux = (int)((W + g->Mx + 2 - g->x_off + g->RW - 1) / g->RW);
    g->nuy = (int)((H + g->My + 2 - g->y_off + g->RH - 1) / g->RH);
    if ((long long)g->nux * g->nuy > (1ll << 24)) return false;
    g->max_stray = 1 << 18;
    g->chk_shrink = chk;
    return true;
}

// TMA descriptors of the unit kernel: one {BW, BH} box per array.  Off-frame elements: zero fill for raw / bias / dark /
// flat (flat = 0 < flat_min: masked), NaN fill for the pre-fused gain (NaN gain: masked).
static bool unit_maps(argus_ctx* c, const FrameArgs& f, int64_t W, int64_t H, const UnitGeom& g) {
    if (!c->encode_tried) {
        c->encode_tried = true;
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qr;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) == cudaSuccess && qr == cudaDriverEntryPointSuccess)
            c->encode_fn = fn;
        else
            (void)cudaGetLastError();
    }
    if (!c->encode_fn) return false;
    const void* key[4] = {f.raw, f.pre ? f.offset : (const void*)f.bias, f.pre ? f.gain : (const void*)f.dark, f.pre ? nullptr : (const void*)f.flat};
    if (memcmp(key, c->umaps_key, sizeof(key)) == 0 && c->umaps_W == W && c->umaps_H == H && c->umaps_bw == g.BW && c->umaps_bh == g.BH &&
        c->umaps_fmt == f.pre)
        return true;
    encode_tiled_fn enc = (encode_tiled_fn)c->encode_fn;
    const int narr = f.pre ? 3 : 4;
    for (int a = 0; a < narr; ++a) {
        const bool half = f.pre == 2 && a > 0;
        const unsigned es = a == 0 ? 2u : (half ? 2u : 4u);
        cuuint64_t dims[2] = {(cuuint64_t)W, (cuuint64_t)H};
        cuuint64_t strides[1] = {(cuuint64_t)W * es};
        cuuint32_t box[2] = {(cuuint32_t)g.BW, (cuuint32_t)g.BH};
        cuuint32_t el[2] = {1, 1};
        const CUtensorMapDataType dt = a == 0 ? CU_TENSOR_MAP_DATA_TYPE_UINT16 : (half ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32);
        const CUtensorMapFloatOOBfill fill = (f.pre && a == 2) ? CU_TENSOR_MAP_FLOAT_OOB_FILL_NAN_REQUEST_ZERO_FMA : CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE;
        CUresult r = enc(&c->umaps.m[a], dt, 2, const_cast<void*>(key[a]), dims, strides, box, el, CU_TENSOR_MAP_INTERLEAVE_NONE,
                         CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, fill);
        if (r != CUDA_SUCCESS) { c->umaps_W = -1; return false; }
    }
    memcpy(c->umaps_key, key, sizeof(key));
    c->umaps_W = W; c->umaps_H = H; c->umaps_bw = g.BW; c->umaps_bh = g.BH; c->umaps_fmt = f.pre;
    return true;
}

// Which kernel runs the planned frame: 2 = image-aligned units, 1 = tile kernel (resample_fast.cuh), 0 = general kernel.
static int choose_path(argus_ctx* c, const FrameArgs& f, bool fused, int kernel, const argus_wcs* wcs, int64_t W, int64_t H, int64_t nside,
                       UnitGeom* ug) {
    c->lz_small = false;
    if (!fused || !c->fast_enabled) return 0;
    if (c->unit_enabled && f.raw && !f.bpm && W % 8 == 0 && W >= 8 && aligned(f.raw, 16) &&
        (f.pre ? (aligned(f.offset, 16) && aligned(f.gain, 16)) : (aligned(f.bias, 16) && aligned(f.dark, 16) && aligned(f.flat, 16)))) {
        DevWcs dw;
        double rho, s_rad;
        // units where the tile kernel cannot run the frame: pre-fused masters, or tiles whose bounding box does not fit its
        // stage somewhere on the frame (HEALPix tiles are wide near the equator and tall in the polar caps); where its
        // boxes fit, the tile kernel is the faster one (0.28 vs 0.33 ms at configs[1]: DESIGN.md 6.6)
        bool tiles_fit = true, tiles_small = false;
        const bool units = make_devwcs(wcs, W, H, nside, &dw, &rho, &s_rad) == ARGUS_OK &&
                           unit_geometry(dw, wcs, W, H, nside, s_rad, kernel, ug, &tiles_fit, &tiles_small, c->unit_margin);
        if (units && (f.pre || !tiles_fit || c->unit_forced) && unit_maps(c, f, W, H, *ug))
            return 2;
        // fine HEALPix grids: every tile's box fits half the Lanczos-3 stage, the tile kernel then runs with two stages (a tile
        // that does not fit after all fails fast_box in the plan and goes to the general kernel)
        c->lz_small = tiles_small && c->lz_small_enabled;
    }
    return fast_maps(c, f, W, H) ? 1 : 0;
}

template <bool COADD>
static int launch_units(argus_ctx* c, int kernel, const UnitGeom& g, const FrameArgs& f, float w_min, float* v, float* wt, long long cap,
                        const CoaddArgs& ca, cudaStream_t st) {
    if (!c->unit_attr_set) {
#define UA(CO, K, M) CUDA_TRY(c, cudaFuncSetAttribute(resample_unit_kernel<CO, K, M>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(UnitSmem<M>)))
        UA(false, 0, 0); UA(true, 0, 0); UA(false, 0, 1); UA(true, 0, 1); UA(false, 0, 2); UA(true, 0, 2);
        UA(false, 1, 0); UA(true, 1, 0); UA(false, 1, 1); UA(true, 1, 1); UA(false, 1, 2); UA(true, 1, 2);
#undef UA
        c->unit_attr_set = true;
    }
    const UnitBuffers& ub = c->slot_ub[c->cur_slot];
    const int grid = c->sm_count * 2;
    CUDA_TRY(c, cudaMemsetAsync(ub.stray_rt, 0, sizeof(int), st));      // run-time hand-overs of the previous call (cached plan)
#define UL(K, M) resample_unit_kernel<COADD, K, M><<<grid, UNIT_THREADS, sizeof(UnitSmem<M>), st>>>(c->umaps, c->pb, ub, g, f, w_min, v, wt, cap, ca)
    if (kernel == ARGUS_BILINEAR) { if (f.pre == 0) UL(0, 0); else if (f.pre == 1) UL(0, 1); else UL(0, 2); }
    else { if (f.pre == 0) UL(1, 0); else if (f.pre == 1) UL(1, 1); else UL(1, 2); }
#undef UL
    // strays, then the plan's slow list (ring / pole tiles, tiles whose cubic does not fit the fixed-point split): general kernel
    if (kernel == ARGUS_BILINEAR) {
        resample_stray_kernel<0, COADD><<<c->sm_count, 256, 0, st>>>(c->dw, c->pb, ub, g.max_stray, f, w_min, v, wt, cap, ca);
        resample_tiles_kernel<0, true, COADD><<<c->sm_count * 2, RS_THREADS, 0, st>>>(c->dw, c->pb, f, w_min, v, wt, cap, ca, 1);
    } else {
        resample_stray_kernel<1, COADD><<<c->sm_count * 4, 256, 0, st>>>(c->dw, c->pb, ub, g.max_stray, f, w_min, v, wt, cap, ca);
        resample_tiles_kernel<1, true, COADD><<<c->sm_count * 2, RS_THREADS, 0, st>>>(c->dw, c->pb, f, w_min, v, wt, cap, ca, 1);
    }
    c->n_launches += 3;
    return ARGUS_OK;
}

template <bool COADD>
static int launch_tiles(argus_ctx* c, int kernel, bool fused, bool use_fast, const FrameArgs& f, int64_t W, int64_t H, float w_min,
                        float* v, float* wt, long long cap, const CoaddArgs& ca, cudaStream_t st) {
    int grid = c->sm_count * 8;
    int slow_only = 0;
    if (use_fast) {
        // TMA-staged hot kernel for every tile that fits a stage; the general kernel takes the rest
        if (!c->fast_attr_set) {
            CUDA_TRY(c, cudaFuncSetAttribute(resample_fast_kernel<false, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FastSmem<0>)));
            CUDA_TRY(c, cudaFuncSetAttribute(resample_fast_kernel<true, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FastSmem<0>)));
            CUDA_TRY(c, cudaFuncSetAttribute(resample_fast_kernel<false, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FastSmem<1>)));
            CUDA_TRY(c, cudaFuncSetAttribute(resample_fast_kernel<true, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FastSmem<1>)));
            CUDA_TRY(c, (cudaFuncSetAttribute(resample_fast_kernel<false, 1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FastSmem<1, 1>))));
            CUDA_TRY(c, (cudaFuncSetAttribute(resample_fast_kernel<true, 1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FastSmem<1, 1>))));
            c->fast_attr_set = true;
        }
        if (kernel == ARGUS_BILINEAR)
            resample_fast_kernel<COADD, 0><<<c->sm_count * FastCfg<0>::CTAS, RF_THREADS, sizeof(FastSmem<0>), st>>>(
                c->maps, c->pb, f, (int)W, (int)H, w_min, v, wt, cap, ca);
        else if (c->pb.fast_cap == FastCfg<1, 1>::CAP)
            resample_fast_kernel<COADD, 1, 1><<<c->sm_count * FastCfg<1, 1>::CTAS, RF_THREADS, sizeof(FastSmem<1, 1>), st>>>(
                c->maps, c->pb, f, (int)W, (int)H, w_min, v, wt, cap, ca);
        else
            resample_fast_kernel<COADD, 1><<<c->sm_count * FastCfg<1>::CTAS, RF_THREADS, sizeof(FastSmem<1>), st>>>(
                c->maps, c->pb, f, (int)W, (int)H, w_min, v, wt, cap, ca);
        c->n_launches++;
        slow_only = 1;
        // slow list: a handful of tiles for bilinear; for Lanczos-3 every box with masked + bright pixels (saturated stars)
        grid = kernel == ARGUS_BILINEAR ? c->sm_count * 2 : c->sm_count * 8;
    }
#define LT(K, F) resample_tiles_kernel<K, F, COADD><<<grid, RS_THREADS, 0, st>>>(c->dw, c->pb, f, w_min, v, wt, cap, ca, slow_only)
    if (kernel == ARGUS_BILINEAR) { if (fused) LT(0, true); else LT(0, false); }
    else { if (fused) LT(1, true); else LT(1, false); }
#undef LT
    c->n_launches++;
    return ARGUS_OK;
}

extern "C" int argus_resample(argus_ctx* c, const argus_frame* frame, const argus_wcs* wcs, int64_t W, int64_t H,
                              int64_t nside, int kernel, float w_min, const int64_t* idx, size_t n, float* value_out,
                              float* weight_out, void* stream) {
    if (!c || !frame || !wcs || !value_out || !weight_out) return ARGUS_ERR_NULL;
    if (kernel != ARGUS_BILINEAR && kernel != ARGUS_LANCZOS3) return ARGUS_ERR_KERNEL;
    if (!aligned(value_out, 4) || !aligned(weight_out, 4) || (idx && !aligned(idx, 8))) return ARGUS_ERR_ALIGN;
    if (n > ((size_t)1 << 40)) return ARGUS_ERR_SHAPE;
    FrameArgs f;
    bool fused;
    int rc = make_frameargs(frame, W, H, &f, &fused);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    CUDA_TRY(c, cudaSetDevice(c->device));
    if (idx) {
        DevWcs dw;
        double rho, s_rad;
        rc = make_devwcs(wcs, W, H, nside, &dw, &rho, &s_rad);
        if (rc) return rc;
        if (n == 0) return ARGUS_OK;
        int nblk = (int)((n + 255) / 256);
        const long long* ip = (const long long*)idx;
#define LL(K, F) resample_list_kernel<K, F><<<nblk, 256, 0, st>>>(dw, f, w_min, ip, (long long)n, value_out, weight_out)
        if (kernel == ARGUS_BILINEAR) { if (fused) LL(0, true); else LL(0, false); }
        else { if (fused) LL(1, true); else LL(1, false); }
#undef LL
        c->n_launches++;
        CUDA_TRY(c, cudaGetLastError());
        return ARGUS_OK;
    }
    int slot = c->prof_n & 255;
    UnitGeom ug;
    const int path = choose_path(c, f, fused, kernel, wcs, W, H, nside, &ug);
    const bool use_fast = path != 0;
    bool replanned = !plan_usable(c, wcs, W, H, nside, !(use_fast && (kernel == ARGUS_BILINEAR || path == 2)), use_fast ? kernel : -1, path == 2 ? &ug : nullptr);
    rc = build_plan(c, wcs, W, H, nside, (long long)n, st, use_fast ? kernel : -1, c->profile ? slot : -1, path == 2 ? &ug : nullptr);
    if (rc) return rc;
    if (c->profile) cudaEventRecord(c->ev[slot][2], st);
    CoaddArgs ca;
    memset(&ca, 0, sizeof(ca));
    if (path == 2) rc = launch_units<false>(c, kernel, ug, f, w_min, value_out, weight_out, (long long)n, ca, st);
    else rc = launch_tiles<false>(c, kernel, fused, use_fast, f, W, H, w_min, value_out, weight_out, (long long)n, ca, st);
    if (rc) return rc;
    mark_slot_read(c, st);
    if (c->profile) { cudaEventRecord(c->ev[slot][3], st); c->ev_plan[slot] = replanned; c->prof_n++; }
    CUDA_TRY(c, cudaGetLastError());
    return ARGUS_OK;
}

// ------------------------------------------------------------------------------- host-buffer variants
// Upload of the HOST raw frame into the next of two device staging sets on the upload stream, ordered after the kernels
// that last read that set; the caller's stream then waits for the upload (and, with outputs, for the previous download
// of the set).  n_out = 0: no output staging (coadd form).
static int host_stage_upload(argus_ctx* c, const argus_frame* frame, int64_t W, int64_t H, size_t n_out, cudaStream_t st,
                             argus_ctx::HostBuf** out_b) {
    if (!c->s_up) {
        CUDA_TRY(c, cudaStreamCreateWithFlags(&c->s_up, cudaStreamNonBlocking));
        CUDA_TRY(c, cudaStreamCreateWithFlags(&c->s_down, cudaStreamNonBlocking));
    }
    argus_ctx::HostBuf& b = c->hb[c->hb_next];
    c->hb_next ^= 1;
    const size_t px = (size_t)W * (size_t)H;
    if (!b.ev_ok) {
        CUDA_TRY(c, cudaEventCreateWithFlags(&b.up, cudaEventDisableTiming));
        CUDA_TRY(c, cudaEventCreateWithFlags(&b.run, cudaEventDisableTiming));
        CUDA_TRY(c, cudaEventCreateWithFlags(&b.down, cudaEventDisableTiming));
        b.ev_ok = true;
    }
    if (b.cap_px < px || b.cap_n < n_out) {      // (re)allocation synchronises: first call per buffer set, or a larger frame
        CUDA_TRY(c, cudaDeviceSynchronize());
        const size_t want_px = b.cap_px > px ? b.cap_px : px, want_n = b.cap_n > n_out ? b.cap_n : n_out;
        if (b.raw) cudaFree(b.raw);
        if (b.val) cudaFree(b.val);
        if (b.wgt) cudaFree(b.wgt);
        b.raw = nullptr; b.val = b.wgt = nullptr; b.cap_px = b.cap_n = 0; b.used = false; b.down_used = false;
        CUDA_TRY(c, cudaMalloc((void**)&b.raw, want_px * sizeof(uint16_t)));
        if (want_n) {
            CUDA_TRY(c, cudaMalloc((void**)&b.val, want_n * sizeof(float)));
            CUDA_TRY(c, cudaMalloc((void**)&b.wgt, want_n * sizeof(float)));
        }
        b.cap_px = want_px; b.cap_n = want_n;
    }
    if (b.used) CUDA_TRY(c, cudaStreamWaitEvent(c->s_up, b.run, 0));
    CUDA_TRY(c, cudaMemcpyAsync(b.raw, frame->raw, px * sizeof(uint16_t), cudaMemcpyHostToDevice, c->s_up));
    CUDA_TRY(c, cudaEventRecord(b.up, c->s_up));
    CUDA_TRY(c, cudaStreamWaitEvent(st, b.up, 0));
    if (n_out && b.down_used) CUDA_TRY(c, cudaStreamWaitEvent(st, b.down, 0));
    *out_b = &b;
    return ARGUS_OK;
}

extern "C" int argus_resample_host(argus_ctx* c, const argus_frame* frame, const argus_wcs* wcs, int64_t W, int64_t H,
                                   int64_t nside, int kernel, float w_min, size_t n, float* value_host, float* weight_host,
                                   void* stream) {
    if (!c || !frame || !wcs || !value_host || !weight_host || !frame->raw) return ARGUS_ERR_NULL;
    if (W < 1 || H < 1 || W > (1 << 20) || H > (1 << 20) || n == 0 || n > ((size_t)1 << 34)) return ARGUS_ERR_SHAPE;
    cudaStream_t st = (cudaStream_t)stream;
    CUDA_TRY(c, cudaSetDevice(c->device));
    argus_ctx::HostBuf* b;
    int rc = host_stage_upload(c, frame, W, H, n, st, &b);
    if (rc) return rc;
    argus_frame fr = *frame;
    fr.raw = b->raw;
    rc = argus_resample(c, &fr, wcs, W, H, nside, kernel, w_min, nullptr, n, b->val, b->wgt, stream);
    if (rc) return rc;
    CUDA_TRY(c, cudaEventRecord(b->run, st));
    b->used = true;
    // download on its own stream
    CUDA_TRY(c, cudaStreamWaitEvent(c->s_down, b->run, 0));
    CUDA_TRY(c, cudaMemcpyAsync(value_host, b->val, n * sizeof(float), cudaMemcpyDeviceToHost, c->s_down));
    CUDA_TRY(c, cudaMemcpyAsync(weight_host, b->wgt, n * sizeof(float), cudaMemcpyDeviceToHost, c->s_down));
    CUDA_TRY(c, cudaEventRecord(b->down, c->s_down));
    b->down_used = true;
    return ARGUS_OK;
}

extern "C" int argus_resample_coadd_host(argus_ctx* c, const argus_frame* frame, const argus_wcs* wcs, int64_t W, int64_t H,
                                         int64_t nside, int kernel, float w_min, const argus_coadd* layout, float* sum,
                                         float* wsum, int64_t* n_skipped_dev, void* stream) {
    if (!c || !frame || !wcs || !frame->raw) return ARGUS_ERR_NULL;
    if (W < 1 || H < 1 || W > (1 << 20) || H > (1 << 20)) return ARGUS_ERR_SHAPE;
    cudaStream_t st = (cudaStream_t)stream;
    CUDA_TRY(c, cudaSetDevice(c->device));
    argus_ctx::HostBuf* b;
    int rc = host_stage_upload(c, frame, W, H, 0, st, &b);
    if (rc) return rc;
    argus_frame fr = *frame;
    fr.raw = b->raw;
    rc = argus_resample_coadd(c, &fr, wcs, W, H, nside, kernel, w_min, layout, sum, wsum, n_skipped_dev, stream);
    if (rc) return rc;
    CUDA_TRY(c, cudaEventRecord(b->run, st));
    b->used = true;
    return ARGUS_OK;
}

// The paper's per-frame product through one call with HOST buffers (PAPER.md:145 16-bit float segment data, :149 / :73 the
// low-resolution map): upload, plan, fused calibrate + resample, footprint list, segment products, download -- 2 bytes
// per footprint pixel leave the device instead of the 8 of value + weight.
extern "C" int argus_reduce_frame_host(argus_ctx* c, const argus_frame* frame, const argus_wcs* wcs, int64_t W, int64_t H,
                                       int64_t nside, int kernel, float w_min, int64_t nside_mini, size_t n, size_t mini_capacity,
                                       uint16_t* seg16_host, int64_t* mini_id_host, float* mini_value_host, float* mini_weight_host,
                                       int64_t* n_mini_host, void* stream) {
    if (!c || !frame || !wcs || !frame->raw || !seg16_host || !mini_id_host || !mini_value_host || !mini_weight_host || !n_mini_host)
        return ARGUS_ERR_NULL;
    if (W < 1 || H < 1 || W > (1 << 20) || H > (1 << 20) || n == 0 || n > ((size_t)1 << 34) || mini_capacity == 0 ||
        mini_capacity > ((size_t)1 << 34))
        return ARGUS_ERR_SHAPE;
    if (!is_pow2(nside_mini) || nside_mini > nside) return ARGUS_ERR_NSIDE;
    cudaStream_t st = (cudaStream_t)stream;
    CUDA_TRY(c, cudaSetDevice(c->device));
    argus_ctx::HostBuf* b;
    int rc = host_stage_upload(c, frame, W, H, n, st, &b);
    if (rc) return rc;
    if (b->cap_prod < n || b->cap_mini < mini_capacity) {
        CUDA_TRY(c, cudaDeviceSynchronize());
        if (b->cap_prod < n) {
            if (b->idx) cudaFree(b->idx);
            if (b->seg16) cudaFree(b->seg16);
            b->idx = nullptr; b->seg16 = nullptr; b->cap_prod = 0;
            CUDA_TRY(c, cudaMalloc((void**)&b->idx, n * sizeof(long long)));
            CUDA_TRY(c, cudaMalloc((void**)&b->seg16, n * sizeof(uint16_t)));
            b->cap_prod = n;
        }
        if (b->cap_mini < mini_capacity) {
            if (b->mini_id) cudaFree(b->mini_id);
            if (b->mini_val) cudaFree(b->mini_val);
            if (b->mini_wgt) cudaFree(b->mini_wgt);
            b->mini_id = nullptr; b->mini_val = b->mini_wgt = nullptr; b->cap_mini = 0;
            CUDA_TRY(c, cudaMalloc((void**)&b->mini_id, mini_capacity * sizeof(long long)));
            CUDA_TRY(c, cudaMalloc((void**)&b->mini_val, mini_capacity * sizeof(float)));
            CUDA_TRY(c, cudaMalloc((void**)&b->mini_wgt, mini_capacity * sizeof(float)));
            b->cap_mini = mini_capacity;
        }
        if (!b->n_mini) CUDA_TRY(c, cudaMalloc((void**)&b->n_mini, sizeof(long long)));
    }
    argus_frame fr = *frame;
    fr.raw = b->raw;
    rc = argus_resample(c, &fr, wcs, W, H, nside, kernel, w_min, nullptr, n, b->val, b->wgt, stream);
    if (rc) return rc;
    plan_write_indices_kernel<<<c->sm_count * 8, 256, 0, st>>>(c->pb, b->idx, (long long)n);
    c->n_launches++;
    mark_slot_read(c, st);
    rc = argus_segment_products(c, nside, nside_mini, (const int64_t*)b->idx, b->val, b->wgt, n, nullptr, 0, nullptr, b->seg16,
                                (int64_t*)b->mini_id, b->mini_val, b->mini_wgt, nullptr, mini_capacity, (int64_t*)b->n_mini, nullptr, stream);
    if (rc) return rc;
    CUDA_TRY(c, cudaEventRecord(b->run, st));
    b->used = true;
    CUDA_TRY(c, cudaStreamWaitEvent(c->s_down, b->run, 0));
    CUDA_TRY(c, cudaMemcpyAsync(seg16_host, b->seg16, n * sizeof(uint16_t), cudaMemcpyDeviceToHost, c->s_down));
    CUDA_TRY(c, cudaMemcpyAsync(mini_id_host, b->mini_id, mini_capacity * sizeof(long long), cudaMemcpyDeviceToHost, c->s_down));
    CUDA_TRY(c, cudaMemcpyAsync(mini_value_host, b->mini_val, mini_capacity * sizeof(float), cudaMemcpyDeviceToHost, c->s_down));
    CUDA_TRY(c, cudaMemcpyAsync(mini_weight_host, b->mini_wgt, mini_capacity * sizeof(float), cudaMemcpyDeviceToHost, c->s_down));
    CUDA_TRY(c, cudaMemcpyAsync(n_mini_host, b->n_mini, sizeof(long long), cudaMemcpyDeviceToHost, c->s_down));
    CUDA_TRY(c, cudaEventRecord(b->down, c->s_down));
    b->down_used = true;
    return ARGUS_OK;
}

extern "C" int argus_host_wait(argus_ctx* c) {
    if (!c) return ARGUS_ERR_NULL;
    CUDA_TRY(c, cudaSetDevice(c->device));
    if (c->s_up) CUDA_TRY(c, cudaStreamSynchronize(c->s_up));
    if (c->s_down) CUDA_TRY(c, cudaStreamSynchronize(c->s_down));
    return ARGUS_OK;
}

static int make_coaddargs(const argus_coadd* lay, int64_t nside, float* sum, float* wsum, int64_t* skipped,
                          CoaddArgs* ca, int* ppt_log2) {
    if (!lay || !lay->tiles || !sum || !wsum) return ARGUS_ERR_NULL;
    if (!is_pow2(nside) || nside < 32 || nside > (1ll << 29)) return ARGUS_ERR_NSIDE;
    if (!is_pow2(lay->nside_tile) || lay->nside_tile > (nside >> ARGUS_TILE_LOG2) || lay->n_tiles < 0) return ARGUS_ERR_SHAPE;
    if (!aligned(lay->tiles, 8) || !aligned(sum, 4) || !aligned(wsum, 4) || (skipped && !aligned(skipped, 8))) return ARGUS_ERR_ALIGN;
    int kk = ilog2(nside) - ilog2(lay->nside_tile);
    ca->tiles = (const long long*)lay->tiles;
    ca->n_tiles = lay->n_tiles;
    ca->shift = 2 * kk - 10;
    ca->sum = sum; ca->wsum = wsum;
    ca->n_skipped = (unsigned long long*)skipped;
    *ppt_log2 = 2 * kk;
    return ARGUS_OK;
}

extern "C" int argus_coadd_accumulate(argus_ctx* c, const argus_coadd* layout, int64_t nside, float* sum, float* wsum,
                                      const int64_t* idx, const float* value, const float* weight, size_t n,
                                      int64_t* n_skipped_dev, void* stream) {
    if (!c || !idx || !value || !weight) return ARGUS_ERR_NULL;
    CoaddArgs ca;
    int ppt_log2;
    int rc = make_coaddargs(layout, nside, sum, wsum, n_skipped_dev, &ca, &ppt_log2);
    if (rc) return rc;
    if (!aligned(idx, 8) || !aligned(value, 4) || !aligned(weight, 4)) return ARGUS_ERR_ALIGN;
    if (n == 0) return ARGUS_OK;
    CUDA_TRY(c, cudaSetDevice(c->device));
    coadd_list_kernel<<<(int)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(ca, ppt_log2, (const long long*)idx, value,
                                                                              weight, (long long)n);
    c->n_launches++;
    CUDA_TRY(c, cudaGetLastError());
    return ARGUS_OK;
}

extern "C" int argus_resample_coadd(argus_ctx* c, const argus_frame* frame, const argus_wcs* wcs, int64_t W, int64_t H,
                                    int64_t nside, int kernel, float w_min, const argus_coadd* layout, float* sum,
                                    float* wsum, int64_t* n_skipped_dev, void* stream) {
    if (!c || !frame || !wcs) return ARGUS_ERR_NULL;
    if (kernel != ARGUS_BILINEAR && kernel != ARGUS_LANCZOS3) return ARGUS_ERR_KERNEL;
    CoaddArgs ca;
    int ppt_log2;
    int rc = make_coaddargs(layout, nside, sum, wsum, n_skipped_dev, &ca, &ppt_log2);
    if (rc) return rc;
    FrameArgs f;
    bool fused;
    rc = make_frameargs(frame, W, H, &f, &fused);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    CUDA_TRY(c, cudaSetDevice(c->device));
    int slot = c->prof_n & 255;
    UnitGeom ug;
    const int path = choose_path(c, f, fused, kernel, wcs, W, H, nside, &ug);
    const bool use_fast = path != 0;
    bool replanned = !plan_usable(c, wcs, W, H, nside, !(use_fast && (kernel == ARGUS_BILINEAR || path == 2)), use_fast ? kernel : -1, path == 2 ? &ug : nullptr);
    rc = build_plan(c, wcs, W, H, nside, -1, st, use_fast ? kernel : -1, c->profile ? slot : -1, path == 2 ? &ug : nullptr);
    if (rc) return rc;
    if (c->profile) cudaEventRecord(c->ev[slot][2], st);
    if (use_fast) {
        coadd_slots_kernel<<<c->sm_count, 256, 0, st>>>(c->pb, ca);
        c->n_launches++;
    }
    if (path == 2) rc = launch_units<true>(c, kernel, ug, f, w_min, nullptr, nullptr, 0, ca, st);
    else rc = launch_tiles<true>(c, kernel, fused, use_fast, f, W, H, w_min, nullptr, nullptr, 0, ca, st);
    if (rc) return rc;
    mark_slot_read(c, st);
    if (c->profile) { cudaEventRecord(c->ev[slot][3], st); c->ev_plan[slot] = replanned; c->prof_n++; }
    CUDA_TRY(c, cudaGetLastError());
    return ARGUS_OK;
}

// ---------------------------------------------------------------------------------------- segment products
extern "C" int argus_segment_products(argus_ctx* c, int64_t nside, int64_t nside_mini, const int64_t* idx,
                                      const float* value, const float* weight, size_t n, const int64_t* targets,
                                      size_t n_targets, const argus_coadd* layout, uint16_t* seg16, int64_t* mini_id,
                                      float* mini_value, float* mini_weight, uint8_t* mini_keep, size_t mini_capacity,
                                      int64_t* n_mini_dev, size_t* n_mini_out, void* stream) {
    if (!c) return ARGUS_ERR_NULL;
    if (n_mini_out) *n_mini_out = 0;
    if (n > 0 && (!idx || !value || !weight)) return ARGUS_ERR_NULL;
    if (n_targets > 0 && !targets) return ARGUS_ERR_NULL;
    if (mini_capacity > 0 && !mini_id) return ARGUS_ERR_NULL;   // the other per-minipix outputs hang off mini_id
    if (mini_capacity == 0 && (seg16 || mini_value || mini_weight || mini_keep)) return ARGUS_ERR_CAPACITY;
    if (!is_pow2(nside) || nside > (1ll << 29)) return ARGUS_ERR_NSIDE;
    if (!is_pow2(nside_mini) || nside_mini > nside) return ARGUS_ERR_NSIDE;
    if (n > (size_t)12 * (size_t)nside * (size_t)nside || mini_capacity > ((size_t)1 << 40)) return ARGUS_ERR_SHAPE;
    if (!aligned(idx, 8) || !aligned(value, 4) || !aligned(weight, 4) || !aligned(targets, 8) || !aligned(seg16, 2) ||
        !aligned(mini_id, 8) || !aligned(mini_value, 4) || !aligned(mini_weight, 4) || !aligned(n_mini_dev, 8))
        return ARGUS_ERR_ALIGN;
    const int shift = 2 * (ilog2(nside) - ilog2(nside_mini));
    SegLayout lay;
    memset(&lay, 0, sizeof(lay));
    if (layout) {
        if (!layout->tiles && layout->n_tiles > 0) return ARGUS_ERR_NULL;
        if (!is_pow2(layout->nside_tile) || layout->nside_tile > nside_mini || layout->n_tiles < 0) return ARGUS_ERR_SHAPE;
        if (!aligned(layout->tiles, 8)) return ARGUS_ERR_ALIGN;
        lay.tiles = (const long long*)layout->tiles;
        lay.n_tiles = layout->n_tiles;
        lay.mini_per_tile_log2 = 2 * (ilog2(nside_mini) - ilog2(layout->nside_tile));
        lay.ppt_log2 = 2 * (ilog2(nside) - ilog2(layout->nside_tile));
    }
    cudaStream_t st = (cudaStream_t)stream;
    CUDA_TRY(c, cudaSetDevice(c->device));
    const size_t n_ctas = (n + SEG_CHUNK - 1) / SEG_CHUNK;
    if (n_ctas > 0x7fffffffull) return ARGUS_ERR_SHAPE;
    // scratch (grown on demand: synchronises the device the first time and when a larger call arrives)
    if (!c->seg.h_n) CUDA_TRY(c, cudaMallocHost((void**)&c->seg.h_n, sizeof(long long)));
    if (c->seg.cap_ctas < n_ctas || !c->seg.ctl) {
        if (c->seg.ctl) { CUDA_TRY(c, cudaDeviceSynchronize()); cudaFree(c->seg.ctl); c->seg.ctl = nullptr; }
        size_t want = align_up(n_ctas + 1, 4096);
        // [2 words: -, n_mini][want chunk offsets, 8 B][want chunk counts, 4 B][want * 128 flag words, 4 B]
        CUDA_TRY(c, cudaMalloc((void**)&c->seg.ctl, 16 + want * (8 + 4 + 4 * (SEG_CHUNK / 32))));
        c->seg.cap_ctas = want;
    }
    long long* seg_offsets = (long long*)(c->seg.ctl + 2);
    unsigned int* seg_counts = (unsigned int*)(seg_offsets + c->seg.cap_ctas);
    unsigned int* seg_bits = seg_counts + c->seg.cap_ctas;
    if (c->seg.cap_mini < mini_capacity || !c->seg.mini_start) {
        if (c->seg.mini_start) { CUDA_TRY(c, cudaDeviceSynchronize()); cudaFree(c->seg.mini_start); c->seg.mini_start = nullptr; }
        size_t want = align_up(mini_capacity + 1, 65536);
        CUDA_TRY(c, cudaMalloc((void**)&c->seg.mini_start, (want + 1) * sizeof(long long)));
        c->seg.cap_mini = want;
    }
    if (n_ctas == 0) {
        CUDA_TRY(c, cudaMemsetAsync(c->seg.ctl, 0, 16, st));
        if (n_mini_dev) CUDA_TRY(c, cudaMemsetAsync(n_mini_dev, 0, sizeof(int64_t), st));
    }
    if (n_ctas > 0) {
        seg_flags_kernel<<<(unsigned)n_ctas, 256, 0, st>>>((const long long*)idx, (long long)n, shift, seg_bits, seg_counts);
        seg_scan_kernel<<<1, 1024, 0, st>>>(seg_counts, (long long)n_ctas, seg_offsets, c->seg.ctl, (long long*)n_mini_dev,
                                            c->seg.mini_start, (long long)mini_capacity, (long long)n);
        c->n_launches += 2;
        if (mini_capacity > 0) {
            seg_heads_kernel<<<(unsigned)((n_ctas + SEG_HEADS_CPB - 1) / SEG_HEADS_CPB), SEG_HEADS_CPB * SEG_CHUNK / 32, 0, st>>>(
                seg_bits, seg_counts, (long long)n_ctas, seg_offsets, (const long long*)idx, shift,
                c->seg.mini_start, (long long*)mini_id, mini_keep, (long long)mini_capacity);
            c->n_launches++;
        }
        if (mini_capacity > 0) {
            if (mini_keep) {
                if (n_targets > 0) {
                    seg_targets_kernel<<<(unsigned)((n_targets + 255) / 256), 256, 0, st>>>(
                        (const long long*)targets, (long long)n_targets, (const long long*)mini_id, c->seg.ctl,
                        (long long)mini_capacity, mini_keep);
                    c->n_launches++;
                }
            }
            if (seg16 || mini_value || mini_weight) {
                const int grid = c->sm_count * 4;
                if (layout && c->seg_raster)
                    seg_products_kernel<2><<<grid, 256, 0, st>>>(c->seg.mini_start, (const long long*)mini_id, mini_keep,
                                                                c->seg.ctl, (long long)mini_capacity, (const long long*)idx,
                                                                value, weight, shift, lay, seg16, mini_value, mini_weight);
                else if (layout)
                    seg_products_kernel<1><<<grid, 256, 0, st>>>(c->seg.mini_start, (const long long*)mini_id, mini_keep,
                                                                c->seg.ctl, (long long)mini_capacity, (const long long*)idx,
                                                                value, weight, shift, lay, seg16, mini_value, mini_weight);
                else
                    seg_products_kernel<0><<<grid, 256, 0, st>>>(c->seg.mini_start, (const long long*)mini_id, mini_keep,
                                                                    c->seg.ctl, (long long)mini_capacity, (const long long*)idx,
                                                                    value, weight, shift, lay, seg16, mini_value, mini_weight);
                c->n_launches++;
            }
        }
        CUDA_TRY(c, cudaGetLastError());
    }
    if (n_mini_out) {
        CUDA_TRY(c, cudaMemcpyAsync(c->seg.h_n, c->seg.ctl + 1, sizeof(long long), cudaMemcpyDeviceToHost, st));
        CUDA_TRY(c, cudaStreamSynchronize(st));
        *n_mini_out = (size_t)*c->seg.h_n;
        if (mini_capacity > 0 && *n_mini_out > mini_capacity) return ARGUS_ERR_CAPACITY;
    }
    return ARGUS_OK;
}

// ------------------------------------------------------------------------- background map + source detection
static int bg_check_cell(int32_t cell) { return (cell == 8 || cell == 16 || cell == 32 || cell == 64) ? ARGUS_OK : ARGUS_ERR_SHAPE; }

extern "C" int argus_background_map(argus_ctx* c, const argus_frame* frame, int64_t W, int64_t H, int32_t cell, int32_t n_min,
                                    float* bkg_out, float* nse_out, float* med_out, float* sig_out, int32_t* ngood_out,
                                    void* stream) {
    if (!c || !frame || !bkg_out || !nse_out) return ARGUS_ERR_NULL;
    if (W < 1 || H < 1 || W > (1 << 20) || H > (1 << 20) || n_min < 0) return ARGUS_ERR_SHAPE;
    if (bg_check_cell(cell)) return ARGUS_ERR_SHAPE;
    if (!aligned(bkg_out, 4) || !aligned(nse_out, 4) || !aligned(med_out, 4) || !aligned(sig_out, 4) || !aligned(ngood_out, 4))
        return ARGUS_ERR_ALIGN;
    FrameArgs f;
    bool fused;
    int rc = make_frameargs(frame, W, H, &f, &fused);
    if (rc) return rc;
    const int64_t GX = (W + cell - 1) / cell, GY = (H + cell - 1) / cell, G = GX * GY;
    if (G > 0x7fffffffll) return ARGUS_ERR_SHAPE;
    cudaStream_t st = (cudaStream_t)stream;
    CUDA_TRY(c, cudaSetDevice(c->device));
    if (c->bg.cap_cells < (size_t)G || !c->bg.cells) {
        if (c->bg.cells) { CUDA_TRY(c, cudaDeviceSynchronize()); cudaFree(c->bg.cells); c->bg.cells = nullptr; }
        size_t want = align_up((size_t)G, 4096);
        CUDA_TRY(c, cudaMalloc((void**)&c->bg.cells, want * 12));
        c->bg.cap_cells = want;
    }
    float* med = med_out ? med_out : c->bg.cells;
    float* sig = sig_out ? sig_out : c->bg.cells + c->bg.cap_cells;
    int* ngood = ngood_out ? (int*)ngood_out : (int*)(c->bg.cells + 2 * c->bg.cap_cells);
    if (fused)
        bg_cells_kernel<true><<<(unsigned)G, BG_THREADS, 0, st>>>(f, (int)W, (int)H, cell, (int)GX, n_min, med, sig, ngood, BgCand{});
    else
        bg_cells_kernel<false><<<(unsigned)G, BG_THREADS, 0, st>>>(f, (int)W, (int)H, cell, (int)GX, n_min, med, sig, ngood, BgCand{});
    bg_filter_kernel<<<(unsigned)((G + 127) / 128), 128, 0, st>>>(med, sig, ngood, (int)GX, (int)GY, n_min, bkg_out, nse_out);
    c->n_launches += 2;
    CUDA_TRY(c, cudaGetLastError());
    return ARGUS_OK;
}

// ---- argus_background_map_static: the same two kernels with the cell scratch in a file-scope device array (no allocation).
// In host code `g_bg_static_cells` is only a host-side stand-in for the symbol, never a device address: the address of the
// array on a device comes from cudaGetSymbolAddress with that device current, once per device (bg_static_address).
// Layout as the context's bg.cells: med [MAX] | sig [MAX] | ngood [MAX] (int bits), 12 bytes per cell.
#define BG_STATIC_MAX_DEVICES 64
static __device__ __align__(256) float g_bg_static_cells[3 * (size_t)ARGUS_BG_STATIC_MAX_CELLS];
static std::mutex g_bg_static_mutex;
static float* g_bg_static_ptr[BG_STATIC_MAX_DEVICES];   // device address of g_bg_static_cells per device, nullptr = not resolved yet

static cudaError_t bg_static_address(float** ptr) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= BG_STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_bg_static_mutex);
    if (!g_bg_static_ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_bg_static_cells);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_bg_static_ptr[dev] = (float*)p;
    }
    *ptr = g_bg_static_ptr[dev];
    return cudaSuccess;
}

extern "C" int argus_background_map_static(const argus_frame* frame, int64_t W, int64_t H, int32_t cell, int32_t n_min,
                                           float* bkg_out, float* nse_out, int32_t* cuda_error_out, void* stream) {
    if (!frame || !bkg_out || !nse_out) return ARGUS_ERR_NULL;
    if (W < 1 || H < 1 || W > (1 << 20) || H > (1 << 20) || n_min < 0) return ARGUS_ERR_SHAPE;
    if (bg_check_cell(cell)) return ARGUS_ERR_SHAPE;
    if (!aligned(bkg_out, 4) || !aligned(nse_out, 4)) return ARGUS_ERR_ALIGN;
    FrameArgs f;
    bool fused;
    int rc = make_frameargs(frame, W, H, &f, &fused);
    if (rc) return rc;
    const int64_t GX = (W + cell - 1) / cell, GY = (H + cell - 1) / cell, G = GX * GY;
    if (G > (int64_t)ARGUS_BG_STATIC_MAX_CELLS) return ARGUS_ERR_CAPACITY;   // the static scratch holds no more cells
    cudaStream_t st = (cudaStream_t)stream;
    float* cells = nullptr;
    cudaError_t e = bg_static_address(&cells);
    if (e == cudaSuccess) {
        float* med = cells;
        float* sig = cells + (size_t)ARGUS_BG_STATIC_MAX_CELLS;
        int* ngood = (int*)(cells + 2 * (size_t)ARGUS_BG_STATIC_MAX_CELLS);
        if (fused)
            bg_cells_kernel<true><<<(unsigned)G, BG_THREADS, 0, st>>>(f, (int)W, (int)H, cell, (int)GX, n_min, med, sig, ngood, BgCand{});
        else
            bg_cells_kernel<false><<<(unsigned)G, BG_THREADS, 0, st>>>(f, (int)W, (int)H, cell, (int)GX, n_min, med, sig, ngood, BgCand{});
        bg_filter_kernel<<<(unsigned)((G + 127) / 128), 128, 0, st>>>(med, sig, ngood, (int)GX, (int)GY, n_min, bkg_out, nse_out);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        if (cuda_error_out) *cuda_error_out = (int32_t)e;
        return ARGUS_ERR_CUDA;
    }
    return ARGUS_OK;
}

// Detection scratch (grown on demand, which synchronises the device): pinned count, control words, per-tile
// (base, count) + offsets, record staging for `capacity` records.
static int det_ensure_scratch(argus_ctx* c, int64_t n_tiles, size_t capacity) {
    if (!c->bg.h_n) CUDA_TRY(c, cudaMallocHost((void**)&c->bg.h_n, sizeof(long long)));
    if (!c->bg.ctl) CUDA_TRY(c, cudaMalloc((void**)&c->bg.ctl, 16));
    if (c->bg.cap_tiles < (size_t)n_tiles || !c->bg.tiles) {
        if (c->bg.tiles) { CUDA_TRY(c, cudaDeviceSynchronize()); cudaFree(c->bg.tiles); c->bg.tiles = nullptr; }
        size_t want = align_up((size_t)n_tiles, 4096);
        CUDA_TRY(c, cudaMalloc((void**)&c->bg.tiles, want * 16));   // tile_info (8 B) | offsets (4 B) | per-band counts (<= one per tile)
        c->bg.cap_tiles = want;
    }
    if (c->bg.cap_tmp < capacity || !c->bg.tmp) {
        if (c->bg.tmp) { CUDA_TRY(c, cudaDeviceSynchronize()); cudaFree(c->bg.tmp); cudaFree(c->bg.ord); c->bg.tmp = nullptr; c->bg.ord = nullptr; }
        size_t want = align_up(capacity + 1, 65536);
        CUDA_TRY(c, cudaMalloc((void**)&c->bg.tmp, want * sizeof(ArgusSourceRec)));
        CUDA_TRY(c, cudaMalloc((void**)&c->bg.ord, want * sizeof(uint2)));
        c->bg.cap_tmp = want;
    }
    return ARGUS_OK;
}

static DetGrid det_grid(const float* bkg, const float* nse, int64_t W, int64_t H, int32_t cell, float k_sigma) {
    DetGrid g;
    g.bkg = bkg; g.nse = nse; g.B = cell;
    g.GX = (int)((W + cell - 1) / cell); g.GY = (int)((H + cell - 1) / cell);
    g.inv_B = 1.0f / (float)cell; g.half = 0.5f * (float)(cell - 1); g.k_sigma = k_sigma;
    return g;
}

// Records -> catalogue order (R-D6), count to the caller (shared by both detection entry points).
static int det_finish(argus_ctx* c, int64_t n_tiles, int64_t tiles_x, int64_t tiles_y, int64_t W, argus_source* out,
                      size_t capacity, int64_t* n_dev, size_t* n_out, cudaStream_t st) {
    unsigned* offsets = (unsigned*)(c->bg.tiles + c->bg.cap_tiles);
    if (capacity > 0)
        det_order_kernel<<<(unsigned)tiles_y, 256, 0, st>>>(c->bg.tiles, offsets, (int)n_tiles, (int)tiles_x, (int)W, offsets + c->bg.cap_tiles,
                                                           c->bg.tmp, c->bg.ord, (ArgusSourceRec*)out, (unsigned)capacity, (long long*)n_dev);
    else
        det_count_kernel<<<1, 1, 0, st>>>(c->bg.ctl, (long long*)n_dev);
    c->n_launches++;
    CUDA_TRY(c, cudaGetLastError());
    if (n_out) {
        CUDA_TRY(c, cudaMemcpyAsync(c->bg.h_n, c->bg.ctl, 8, cudaMemcpyDeviceToHost, st));
        CUDA_TRY(c, cudaStreamSynchronize(st));
        *n_out = (size_t)(((unsigned long long)*c->bg.h_n) & 0xffffffffull);     // ctl[0]: the running total of the tile kernels
        if (capacity > 0 && *n_out > capacity) return ARGUS_ERR_CAPACITY;
    }
    return ARGUS_OK;
}

// ctl and the per-band counts start at zero
static int det_clear(argus_ctx* c, int64_t tiles_y, cudaStream_t st) {
    unsigned* band_cnt = (unsigned*)(c->bg.tiles + c->bg.cap_tiles) + c->bg.cap_tiles;
    CUDA_TRY(c, cudaMemsetAsync(c->bg.ctl, 0, 16, st));
    CUDA_TRY(c, cudaMemsetAsync(band_cnt, 0, (size_t)tiles_y * 4, st));
    return ARGUS_OK;
}

extern "C" int argus_detect_sources(argus_ctx* c, const argus_frame* frame, int64_t W, int64_t H, int32_t cell,
                                    const float* bkg, const float* nse, float k_sigma, argus_source* out, size_t capacity,
                                    int64_t* n_dev, size_t* n_out, void* stream) {
    if (!c) return ARGUS_ERR_NULL;
    if (n_out) *n_out = 0;
    if (!frame || !bkg || !nse || (capacity > 0 && !out)) return ARGUS_ERR_NULL;
    if (W < 1 || H < 1 || W > (1 << 20) || H > (1 << 20) || capacity > 0x7fffffffull) return ARGUS_ERR_SHAPE;
    if (bg_check_cell(cell) || !(k_sigma >= 0.0f) || !(k_sigma < INFINITY)) return ARGUS_ERR_SHAPE;
    if (!aligned(bkg, 4) || !aligned(nse, 4) || !aligned(out, 16) || !aligned(n_dev, 8)) return ARGUS_ERR_ALIGN;
    FrameArgs f;
    bool fused;
    int rc = make_frameargs(frame, W, H, &f, &fused);
    if (rc) return rc;
    const int64_t tiles_x = (W + DET_TW - 1) / DET_TW, tiles_y = (H + DET_TH - 1) / DET_TH, n_tiles = tiles_x * tiles_y;
    if (n_tiles > 0x7fffffffll) return ARGUS_ERR_SHAPE;
    cudaStream_t st = (cudaStream_t)stream;
    CUDA_TRY(c, cudaSetDevice(c->device));
    rc = det_ensure_scratch(c, n_tiles, capacity);
    if (rc) return rc;
    const DetGrid g = det_grid(bkg, nse, W, H, cell, k_sigma);
    rc = det_clear(c, tiles_y, st);
    if (rc) return rc;
    unsigned* band_cnt = (unsigned*)(c->bg.tiles + c->bg.cap_tiles) + c->bg.cap_tiles;
    if (fused)
        det_tiles_kernel<true><<<(unsigned)n_tiles, 256, 0, st>>>(f, (int)W, (int)H, g, (int)tiles_x, c->bg.tmp, (unsigned)capacity,
                                                               c->bg.tiles, c->bg.ctl, band_cnt);
    else
        det_tiles_kernel<false><<<(unsigned)n_tiles, 256, 0, st>>>(f, (int)W, (int)H, g, (int)tiles_x, c->bg.tmp, (unsigned)capacity,
                                                                c->bg.tiles, c->bg.ctl, band_cnt);
    c->n_launches++;
    return det_finish(c, n_tiles, tiles_x, tiles_y, W, out, capacity, n_dev, n_out, st);
}

// Background map + detection in one call: the candidates of every tile are collected while the cell statistics are formed,
// so the frame is read once; results identical to argus_background_map followed by argus_detect_sources.
extern "C" int argus_detect_frame(argus_ctx* c, const argus_frame* frame, int64_t W, int64_t H, int32_t cell, int32_t n_min,
                                  float k_sigma, float* bkg_out, float* nse_out, argus_source* out, size_t capacity,
                                  int64_t* n_dev, size_t* n_out, void* stream) {
    if (!c) return ARGUS_ERR_NULL;
    if (n_out) *n_out = 0;
    if (!frame || !bkg_out || !nse_out || (capacity > 0 && !out)) return ARGUS_ERR_NULL;
    if (W < 1 || H < 1 || W > (1 << 20) || H > (1 << 20) || n_min < 0 || capacity > 0x7fffffffull) return ARGUS_ERR_SHAPE;
    if (bg_check_cell(cell) || !(k_sigma >= 0.0f) || !(k_sigma < INFINITY)) return ARGUS_ERR_SHAPE;
    if (!aligned(bkg_out, 4) || !aligned(nse_out, 4) || !aligned(out, 16) || !aligned(n_dev, 8)) return ARGUS_ERR_ALIGN;
    FrameArgs f;
    bool fused;
    int rc = make_frameargs(frame, W, H, &f, &fused);
    if (rc) return rc;
    const int64_t GX = (W + cell - 1) / cell, GY = (H + cell - 1) / cell, G = GX * GY;
    const int64_t tiles_x = (W + DET_TW - 1) / DET_TW, tiles_y = (H + DET_TH - 1) / DET_TH, n_tiles = tiles_x * tiles_y;
    if (G > 0x7fffffffll || n_tiles > 0x7fffffffll) return ARGUS_ERR_SHAPE;
    cudaStream_t st = (cudaStream_t)stream;
    CUDA_TRY(c, cudaSetDevice(c->device));
    if (c->bg.cap_cells < (size_t)G || !c->bg.cells) {
        if (c->bg.cells) { CUDA_TRY(c, cudaDeviceSynchronize()); cudaFree(c->bg.cells); c->bg.cells = nullptr; }
        size_t want = align_up((size_t)G, 4096);
        CUDA_TRY(c, cudaMalloc((void**)&c->bg.cells, want * 12));
        c->bg.cap_cells = want;
    }
    // candidate scratch: cut [G] | cnt [n_lists] | fb_count (4 words) | fb_list [n_tiles] | list [n_lists][cap] u16
    const size_t n_lists = (cell == 64 ? 2 : 1) * (size_t)G, Gp = align_up((size_t)G, 64), Lp = align_up(n_lists, 64), Tp = align_up((size_t)n_tiles, 64);
    const size_t cand_bytes = (Gp + Lp + 4 + Tp) * 4 + Lp * (size_t)det_cand_cap(cell) * 2;
    if (c->bg.cap_cand < cand_bytes || !c->bg.cand) {
        if (c->bg.cand) { CUDA_TRY(c, cudaDeviceSynchronize()); cudaFree(c->bg.cand); c->bg.cand = nullptr; }
        const size_t want = align_up(cand_bytes, (size_t)1 << 20);
        CUDA_TRY(c, cudaMalloc((void**)&c->bg.cand, want));
        c->bg.cap_cand = want;
    }
    rc = det_ensure_scratch(c, n_tiles, capacity);
    if (rc) return rc;
    BgCand cd;
    cd.cut = (float*)c->bg.cand;
    cd.cnt = (unsigned*)(cd.cut + Gp);
    unsigned* fb_count = cd.cnt + Lp;
    unsigned* fb_list = fb_count + 4;
    cd.list = (unsigned short*)(fb_list + Tp);
    // the cut must leave room below the threshold for the proof of det_cand_kernel and keep the lists short
    cd.kappa = fmaxf(k_sigma - 2.0f, 2.5f);
    float* med = c->bg.cells;
    float* sig = c->bg.cells + c->bg.cap_cells;
    int* ngood = (int*)(c->bg.cells + 2 * c->bg.cap_cells);
    const DetGrid g = det_grid(bkg_out, nse_out, W, H, cell, k_sigma);
    rc = det_clear(c, tiles_y, st);
    if (rc) return rc;
    unsigned* band_cnt = (unsigned*)(c->bg.tiles + c->bg.cap_tiles) + c->bg.cap_tiles;
    CUDA_TRY(c, cudaMemsetAsync(fb_count, 0, 16, st));
    const unsigned fb_grid = (unsigned)std::min<int64_t>(n_tiles, (int64_t)c->sm_count * 8);
    if (fused) {
        bg_cells_kernel<true, true><<<(unsigned)G, BG_THREADS, 0, st>>>(f, (int)W, (int)H, cell, (int)GX, n_min, med, sig, ngood, cd);
        bg_filter_kernel<<<(unsigned)((G + 127) / 128), 128, 0, st>>>(med, sig, ngood, (int)GX, (int)GY, n_min, bkg_out, nse_out);
        det_cand_kernel<true><<<(unsigned)((n_tiles + 7) / 8), 256, 0, st>>>(f, (int)W, (int)H, g, (int)tiles_x, (int)n_tiles, cd.cnt, cd.list,
                                                                             cd.cut, c->bg.tmp, (unsigned)capacity, c->bg.tiles, c->bg.ctl,
                                                                             band_cnt, fb_list, fb_count);
        det_tiles_list_kernel<true><<<fb_grid, 256, 0, st>>>(f, (int)W, (int)H, g, (int)tiles_x, c->bg.tmp, (unsigned)capacity, c->bg.tiles,
                                                             c->bg.ctl, band_cnt, fb_list, fb_count);
    } else {
        bg_cells_kernel<false, true><<<(unsigned)G, BG_THREADS, 0, st>>>(f, (int)W, (int)H, cell, (int)GX, n_min, med, sig, ngood, cd);
        bg_filter_kernel<<<(unsigned)((G + 127) / 128), 128, 0, st>>>(med, sig, ngood, (int)GX, (int)GY, n_min, bkg_out, nse_out);
        det_cand_kernel<false><<<(unsigned)((n_tiles + 7) / 8), 256, 0, st>>>(f, (int)W, (int)H, g, (int)tiles_x, (int)n_tiles, cd.cnt, cd.list,
                                                                              cd.cut, c->bg.tmp, (unsigned)capacity, c->bg.tiles, c->bg.ctl,
                                                                              band_cnt, fb_list, fb_count);
        det_tiles_list_kernel<false><<<fb_grid, 256, 0, st>>>(f, (int)W, (int)H, g, (int)tiles_x, c->bg.tmp, (unsigned)capacity, c->bg.tiles,
                                                              c->bg.ctl, band_cnt, fb_list, fb_count);
    }
    c->n_launches += 4;
    c->bg.last_fb = fb_count;
    return det_finish(c, n_tiles, tiles_x, tiles_y, W, out, capacity, n_dev, n_out, st);
}

extern "C" int argus_detect_frame_info(argus_ctx* c, int64_t* n_full_tiles, void* stream) {
    if (!c || !n_full_tiles) return ARGUS_ERR_NULL;
    *n_full_tiles = 0;
    if (!c->bg.last_fb) return ARGUS_ERR_STATE;
    CUDA_TRY(c, cudaSetDevice(c->device));
    unsigned v = 0;
    CUDA_TRY(c, cudaMemcpyAsync(&v, c->bg.last_fb, 4, cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    CUDA_TRY(c, cudaStreamSynchronize((cudaStream_t)stream));
    *n_full_tiles = (int64_t)v;
    return ARGUS_OK;
}

// ------------------------------------------------------------------------- direct image subtraction per tile (8(f).3)
extern "C" int argus_subtract_tiles(argus_ctx* c, const argus_coadd* layout, int64_t nside, const float* sci_sum,
                                    const float* sci_wsum, const float* ref_sum, const float* ref_wsum,
                                    const argus_subtract_params* prm, float* diff_out, float* sig_out, float* alpha_out,
                                    float* beta_out, int32_t* nvalid_out, argus_transient* cat_out, size_t capacity,
                                    int64_t* n_dev, size_t* n_out, void* stream) {
    if (!c) return ARGUS_ERR_NULL;
    if (n_out) *n_out = 0;
    if (!layout || !prm || (capacity > 0 && !cat_out)) return ARGUS_ERR_NULL;
    if (layout->n_tiles > 0 && (!layout->tiles || !sci_sum || !sci_wsum || !ref_sum || !ref_wsum || !diff_out)) return ARGUS_ERR_NULL;
    if (!is_pow2(nside) || nside < 32 || nside > (1ll << 29)) return ARGUS_ERR_NSIDE;
    if (!is_pow2(layout->nside_tile) || layout->nside_tile > (nside >> ARGUS_TILE_LOG2) || layout->n_tiles < 0) return ARGUS_ERR_SHAPE;
    if (prm->match != ARGUS_SUB_MATCH_NONE && prm->match != ARGUS_SUB_MATCH_AFFINE) return ARGUS_ERR_SHAPE;
    if (prm->n_min < 2 || !(prm->sci_wmin > 0.f) || !(prm->ref_wmin > 0.f) || !(prm->sci_wmin < INFINITY) || !(prm->ref_wmin < INFINITY) ||
        !(prm->read_noise > 0.f) || !(prm->read_noise < INFINITY) || !(prm->gain > 0.f) || !(prm->gain < INFINITY) ||
        !(prm->k_sigma >= 0.f) || !(prm->k_sigma < INFINITY) || capacity > 0x7fffffffull)
        return ARGUS_ERR_SHAPE;
    if (!aligned(sci_sum, 16) || !aligned(sci_wsum, 16) || !aligned(ref_sum, 16) || !aligned(ref_wsum, 16) || !aligned(diff_out, 16) ||
        !aligned(sig_out, 16) || !aligned(alpha_out, 4) || !aligned(beta_out, 4) || !aligned(nvalid_out, 4) || !aligned(cat_out, 16) ||
        !aligned(n_dev, 8) || !aligned(layout->tiles, 8))
        return ARGUS_ERR_ALIGN;
    const int side_log2 = ilog2(nside) - ilog2(layout->nside_tile);     // >= 5
    if (side_log2 > 15) return ARGUS_ERR_SHAPE;
    const long long ppt = 1ll << (2 * side_log2);
    const long long n_tiles = layout->n_tiles, n_blocks = n_tiles * (ppt / SUB_BLOCK);
    if (n_blocks > 0x7fffffffll) return ARGUS_ERR_SHAPE;
    cudaStream_t st = (cudaStream_t)stream;
    CUDA_TRY(c, cudaSetDevice(c->device));
    if (!c->sub.h_n) CUDA_TRY(c, cudaMallocHost((void**)&c->sub.h_n, sizeof(long long)));
    if (!c->sub.ctl) CUDA_TRY(c, cudaMalloc((void**)&c->sub.ctl, 16));
    if (c->sub.cap_tiles < (size_t)n_tiles || !c->sub.fit) {
        if (c->sub.fit) { CUDA_TRY(c, cudaDeviceSynchronize()); cudaFree(c->sub.fit); cudaFree(c->sub.partial); c->sub.fit = nullptr; c->sub.partial = nullptr; }
        size_t want = align_up((size_t)n_tiles + 1, 256);
        CUDA_TRY(c, cudaMalloc((void**)&c->sub.fit, want * sizeof(float2)));
        CUDA_TRY(c, cudaMalloc((void**)&c->sub.partial, want * SUB_SPLIT_MAX * 5 * sizeof(double)));
        c->sub.cap_tiles = want;
    }
    if (c->sub.cap_blocks < (size_t)n_blocks || !c->sub.blocks) {
        if (c->sub.blocks) { CUDA_TRY(c, cudaDeviceSynchronize()); cudaFree(c->sub.blocks); c->sub.blocks = nullptr; }
        size_t want = align_up((size_t)n_blocks + 1, 4096);
        CUDA_TRY(c, cudaMalloc((void**)&c->sub.blocks, want * 12));
        c->sub.cap_blocks = want;
    }
    if (c->sub.cap_tmp < capacity || !c->sub.tmp) {
        if (c->sub.tmp) { CUDA_TRY(c, cudaDeviceSynchronize()); cudaFree(c->sub.tmp); c->sub.tmp = nullptr; }
        size_t want = align_up(capacity + 1, 65536);
        CUDA_TRY(c, cudaMalloc((void**)&c->sub.tmp, want * sizeof(ArgusTransientRec)));
        c->sub.cap_tmp = want;
    }
    unsigned* offsets = (unsigned*)(c->sub.blocks + c->sub.cap_blocks);
    SubParams p;
    p.match = prm->match; p.n_min = prm->n_min; p.sci_wmin = prm->sci_wmin; p.ref_wmin = prm->ref_wmin;
    p.rn2 = prm->read_noise * prm->read_noise; p.inv_gain = 1.0f / prm->gain; p.k_sigma = prm->k_sigma;
    CUDA_TRY(c, cudaMemsetAsync(c->sub.ctl, 0, 16, st));
    if (n_tiles == 0) {
        if (n_dev) CUDA_TRY(c, cudaMemsetAsync(n_dev, 0, sizeof(int64_t), st));
        if (n_out) CUDA_TRY(c, cudaStreamSynchronize(st));
        return ARGUS_OK;
    }
    // statistics pass only when something needs it (the affine fit, or the count of valid pixels)
    const int have_stats = (prm->match == ARGUS_SUB_MATCH_AFFINE || nvalid_out) ? 1 : 0;
    int split = (int)(ppt / 8192);
    if (split < 1) split = 1;
    if (split > SUB_SPLIT_MAX) split = SUB_SPLIT_MAX;
    // The affine match needs every valid pixel of a tile before the first difference can be formed: two passes over the inputs.
    // (Tried: tiles in chunks of 12 / 24 whose inputs fit L2, statistics -> fit -> difference per chunk, so that the second pass
    // reads from L2: 0.95 / 0.78 ms against 0.54 ms for one chunk -- 18 / 9 times three small launches with their tails cost
    // more than the saved HBM reads.  The kernels keep their chunk arguments; one chunk is used.)
    const long long bpt = ppt / SUB_BLOCK;
    const long long chunk = n_tiles;
    if (have_stats && chunk * split > 0x7fffffffll) return ARGUS_ERR_SHAPE;
    for (long long t0 = 0; t0 < n_tiles; t0 += chunk) {
        const long long t1 = t0 + chunk < n_tiles ? t0 + chunk : n_tiles;
        if (have_stats) {
            sub_stats_kernel<<<(unsigned)((t1 - t0) * split), 256, 0, st>>>(sci_sum, sci_wsum, ref_sum, ref_wsum, ppt, split, t0, p, c->sub.partial);
            c->n_launches++;
        }
        sub_fit_kernel<<<(unsigned)((t1 - t0 + 127) / 128), 128, 0, st>>>(c->sub.partial, t0, t1, split, p, have_stats, c->sub.fit, alpha_out,
                                                                         beta_out, (int*)nvalid_out);
        const long long nb = (t1 - t0) * bpt;
        long long grid = nb < (long long)c->sm_count * 32 ? nb : (long long)c->sm_count * 32;
        sub_tiles_kernel<<<(unsigned)grid, 256, 0, st>>>(sci_sum, sci_wsum, ref_sum, ref_wsum, (const long long*)layout->tiles, ppt, side_log2,
                                                        t0 * bpt, t1 * bpt, p, c->sub.fit, diff_out, sig_out, c->sub.tmp, (unsigned)capacity,
                                                        c->sub.blocks, c->sub.ctl);
        c->n_launches += 2;
    }
    det_scan_kernel<<<1, 1024, 0, st>>>(c->sub.blocks, (int)n_blocks, offsets, c->sub.ctl, (long long*)n_dev);
    c->n_launches += 1;
    if (capacity > 0) {
        sub_gather_kernel<<<(unsigned)((n_blocks + 7) / 8), 256, 0, st>>>(c->sub.blocks, offsets, n_blocks, c->sub.tmp,
                                                                        (ArgusTransientRec*)cat_out, (unsigned)capacity);
        c->n_launches++;
    }
    CUDA_TRY(c, cudaGetLastError());
    if (n_out) {
        CUDA_TRY(c, cudaMemcpyAsync(c->sub.h_n, c->sub.ctl, 8, cudaMemcpyDeviceToHost, st));
        CUDA_TRY(c, cudaStreamSynchronize(st));
        *n_out = (size_t)(((unsigned long long)*c->sub.h_n) >> 32);     // ctl[1]
        if (capacity > 0 && *n_out > capacity) return ARGUS_ERR_CAPACITY;
    }
    return ARGUS_OK;
}
