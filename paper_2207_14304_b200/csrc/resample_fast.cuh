// resample_fast.cuh -- A2..A5 (+A6) fused, bilinear or Lanczos-3, TMA-staged: the hot kernel of the path.
//
// Persistent CTAs (bilinear: 2 per SM, 2 stages; Lanczos-3: 3 per SM, 1 stage), 8 consumer warps + 1 producer warp, one
// 32x32 output tile (1024 consecutive nested indices) per iteration, tiles dealt round-robin in ascending order:
//   producer  (software-pipelined) reads the tile's FastRec, issues one cp.async.bulk.tensor (TMA) per array (raw u16,
//             bias, dark, flat f32) for the tile's source bounding box into a free stage -- out-of-frame elements
//             arrive as zeros (flat = 0 < flat_min => masked), so no bounds logic exists anywhere -- writes the tile
//             descriptor (record, output offset, per-column Horner coefficients, membership mask of border tiles) and
//             completes the stage's mbarrier with arrive.expect_tx.  Loads run one to two tiles ahead of the consumers.
//   consumers wait on the mbarrier, calibrate the staged box ONCE: shared -> registers, a barrier, then
//             the float32 box overwrites the stage in place with a bank-conflict-free pitch (masked pixels as NaN);
//             gather: coordinates from the tile polynomial (exact integer linear part + FP32 remainder, common.cuh),
//             2x2 or 6x6 taps, value + weight stores of 32 consecutive floats per warp -- or the coadd
//             read-modify-write; every thread then releases the stage (mbarrier arrive).
// Tiles that do not fit a stage, belt/cap-ring and pole tiles are left to resample_tiles_kernel (the plan's slow list);
// the Lanczos-3 variant appends tiles with masked + bright pixels to that list at run time (FP64 path).
#pragma once
#include <cuda.h>

#include "common.cuh"
#include "plan.cuh"
#include "resample.cuh"

#ifndef RF_CONSUMERS
#define RF_CONSUMERS 256                 // threads of one consumer group (one output tile at a time): 256 or 512
#endif
#define RF_NQ (ARGUS_TILE_PIX / RF_CONSUMERS)   // output pixels per thread
#define RF_GROUPS 1                      // consumer groups per CTA, tiles dealt round-robin
#define RF_THREADS (RF_GROUPS * RF_CONSUMERS + 32)

// Per interpolation kernel (and variant): stage capacity, stages per CTA, CTAs per SM, register cap.
//   bilinear            : 2 stages x 50 KB, 2 CTAs / SM, 80 registers (leaves room for a plan CTA beside it, argus_api.cu)
//   Lanczos-3           : the gather dominates (36 taps, 12 kernel weights per pixel): 1 stage x 64.5 KB calibrated in place,
//                         3 CTAs / SM hide one another's stage fills
//   Lanczos-3, VAR = 1  : frames whose tiles all fit a 48 x 48 box (fine HEALPix grids: nside 2^18 at configs[4]'s pixel
//                         scale), chosen on the host from the WCS: 2 stages x 32 KB in the same shared memory, so a CTA's
//                         next box lands while it gathers
#define FAST_CAP_PX_LZ_SMALL 2304         // Lanczos-3 on fine grids (every box at most 48 x 48 pixels), 2 stages
#define RF_LZ_BIG_ADU 1500.0f              // Lanczos-3: a box with masked AND brighter pixels goes to the FP64 kernel
template <int KERNEL, int VAR = 0> struct FastCfg;
//   SPLIT (one-stage Lanczos-3): the calibrated box overwrites bias + a pad of its own, so raw / dark / flat are dead once
//                         the calibration has read them: the producer refills them for the CTA's next tile during the
//                         gather, and only the bias box (18 of 64.5 KB, prefetched into L2) is loaded after it
#ifndef RF_LZ_SPLIT
#define RF_LZ_SPLIT 1
#endif
#ifndef RF_SCHED_DYNAMIC
#define RF_SCHED_DYNAMIC 1               // 1: Lanczos-3 tiles claimed from a counter instead of dealt round-robin; 2: bilinear too
#endif
template <> struct FastCfg<0, 0> { static constexpr int CAP = FAST_CAP_PX, STAGES = 2, CTAS = 2, TL = 0, TR = 1, CALBUF = 0, REGS = 80, SPLIT = 0; };
template <> struct FastCfg<1, 0> { static constexpr int CAP = FAST_CAP_PX_LZ, STAGES = 1, CTAS = 3, TL = 2, TR = 3, CALBUF = 0, REGS = 72, SPLIT = RF_LZ_SPLIT; };
template <> struct FastCfg<1, 1> { static constexpr int CAP = FAST_CAP_PX_LZ_SMALL, STAGES = 2, CTAS = 3, TL = 2, TR = 3, CALBUF = 0, REGS = 72, SPLIT = 0; };

struct FastMaps {
    CUtensorMap m[4][5][4];   // [height class][width class][raw, bias, dark, flat]; box = (40 + 8 w) x (48 + 8 h)
};

struct __align__(16) FastDesc {
    FastRec r;
    long long off;       // output position of the tile's first pixel
    long long cslot;     // coadd slot of the tile's first pixel, -1 = tile absent from the layout
    int t;               // index of the tile in the plan
    int pad[3];
    float4 tab[32][2];   // per pixel column u: {Ax, Bx, Cx, Ay}, {By, Cy, -, -}: S-dependent Horner coefficients
    unsigned mask[32];   // TC_BORDER: membership bits
    int pref[32];        //            exclusive prefix of popc(mask)
};

// One stage: the raw + master boxes as the TMA delivers them (dense, pitch = box width).  After the consumers have
// read them into registers, the calibrated box overwrites the stage from `bias` on (pitch 8 or 24 mod 32 floats,
// up to CAP * 9/8 floats = bias + the head of dark; with PAD = CAP / 8 the tail lands in a pad of its own instead).
template <int CAP, int PAD = 32>
struct __align__(128) FastStage {
    unsigned short raw[CAP];
    float bias[CAP];
    float calpad[PAD];
    float dark[CAP];
    float flat[CAP];
};
template <int KERNEL, int VAR = 0>
struct __align__(128) FastSmem {
    typedef FastStage<FastCfg<KERNEL, VAR>::CAP, FastCfg<KERNEL, VAR>::SPLIT ? FastCfg<KERNEL, VAR>::CAP / 8 : 32> Stage;
    Stage stage[FastCfg<KERNEL, VAR>::STAGES];
    float calbuf[FastCfg<KERNEL, VAR>::CALBUF > 0 ? FastCfg<KERNEL, VAR>::CALBUF : 4];   // separate calibrated box (Lanczos-3)
    FastDesc desc[2];                                    // tile k uses descriptor k & 1 and stage k % STAGES
    unsigned long long full[2];                          // descriptor written and TMA bytes landed (1 arrival + tx)
    unsigned long long empty[FastCfg<KERNEL, VAR>::STAGES];   // all consumers are done with the stage (RF_CONSUMERS arrivals)
    unsigned long long empty_a;                          // SPLIT: all consumers have read raw / dark / flat of the stage
};

// ---------------------------------------------------------------------------------- PTX wrappers
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* b, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long* b, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* b, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(b)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_prefetch_2d(const CUtensorMap* map, int x, int y) {
    asm volatile("cp.async.bulk.prefetch.tensor.2d.L2.global.tile [%0, {%1, %2}];" ::"l"(map), "r"(x), "r"(y) : "memory");
}
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, int x, int y, unsigned long long* bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(
            smem_u32(dst)),
        "l"(map), "r"(smem_u32(bar)), "r"(x), "r"(y)
        : "memory");
}
// named barrier 1 over the consumer threads, with an OR reduction of a predicate
template <int ID>
__device__ __forceinline__ int bar_sync_or(int pred) {
    int r;
    asm volatile(
        "{\n"
        ".reg .pred p, q;\n"
        "setp.ne.s32 p, %1, 0;\n"
        "barrier.cta.red.or.pred q, %3, %2, p;\n"
        "selp.s32 %0, 1, 0, q;\n"
        "}\n"
        : "=r"(r)
        : "r"(pred), "n"(RF_CONSUMERS), "n"(ID)
        : "memory");
    return r;
}
template <int ID>
__device__ __forceinline__ void bar_sync() {
    asm volatile("barrier.cta.sync %1, %0;" ::"n"(RF_CONSUMERS), "n"(ID) : "memory");
}
// named barrier 1 + group over the threads of one consumer group (ids must be immediates: a register id makes
// ptxas reserve all 16 barriers)
__device__ __forceinline__ int consumers_sync_or(int group, int pred) {
    return group == 0 ? bar_sync_or<1>(pred) : (group == 1 ? bar_sync_or<2>(pred) : bar_sync_or<3>(pred));
}
__device__ __forceinline__ void consumers_sync(int group) {
    if (group == 0) bar_sync<1>(); else if (group == 1) bar_sync<2>(); else bar_sync<3>();
}

// ------------------------------------------------------------------------------------ coordinates
// ceil(2^20 / bw4) for the sixteen box widths 40 + 8 wc (bw4 = 10 + 2 wc float4 items per row)
#define RF_MAGIC_(wc) ((1048576u + (10u + 2u * (wc)) - 1u) / (10u + 2u * (wc)))
__device__ __constant__ unsigned RF_ROW_MAGIC[16] = {RF_MAGIC_(0), RF_MAGIC_(1), RF_MAGIC_(2), RF_MAGIC_(3), RF_MAGIC_(4), RF_MAGIC_(5),
                                                     RF_MAGIC_(6), RF_MAGIC_(7), RF_MAGIC_(8), RF_MAGIC_(9), RF_MAGIC_(10), RF_MAGIC_(11),
                                                     RF_MAGIC_(12), RF_MAGIC_(13), RF_MAGIC_(14), RF_MAGIC_(15)};
struct FastAxis {
    float A0, A1, B0, B1, C0, C1, c9;   // Horner in T; index = S variant (pixel column u or u + 16)
    int lin;                            // c0 + a*s0 + b*t0
    int da, db;                         // 32 a, 32 b: steps to u + 16 / v + 16
};
// Pixel Q of a thread is Morton index gt + RF_CONSUMERS * Q.  With 256 threads bit 8 (Q & 1) moves the pixel 16
// columns (S + 1) and bit 9 (Q >> 1) 16 rows (T + 1); with 512 threads Q only moves rows.  Position in 2^-22 px.
template <int Q>
__device__ __forceinline__ int fast_axis_eval(const FastAxis& ax, float T0, float T1) {
    constexpr bool CV = (RF_CONSUMERS == 256) && (Q & 1);                 // column variant
    constexpr bool RV = (RF_CONSUMERS == 256) ? (Q >> 1) != 0 : Q != 0;   // row variant
    const float T = RV ? T1 : T0;
    const float h = fmaf(T, fmaf(T, fmaf(T, ax.c9, CV ? ax.C1 : ax.C0), CV ? ax.B1 : ax.B0), CV ? ax.A1 : ax.A0);
    return ax.lin + (CV ? ax.da : 0) + (RV ? ax.db : 0) + __float_as_int(h);
}
__device__ __forceinline__ float fast_frac(int xf) {
    // 24 fraction bits: the upper 23 go into the mantissa of 2^23 + m, one FMA brings them to [0, 1)
    return fmaf(__uint_as_float((((unsigned)xf >> 1) & 0x7fffffu) | 0x4B000000u), 1.1920928955078125e-07f, -1.0f);
}

// ------------------------------------------------------------------------------------ interpolation
// Lanczos-3 weights of the six taps at offsets t_q = f + 2 - q (q = 0..5) for the fraction f in [0, 1), UP TO A COMMON
// FACTOR: L(t) = sin(pi t) sin(pi t / 3) * 3 / (pi t)^2, and sin(pi t_q) = (-1)^q sin(pi f) is the same for all six
// taps up to sign, so it cancels in value = sum(k c) / sum(k) and is never computed.  k_q = +-sin(pi t_q / 3) / t_q^2.
// FP32 with bounded RELATIVE error (~2e-7) on every weight, which is what the value tolerance needs next to bright
// taps: every argument is reduced EXACTLY before any rounding (f is a multiple of 2^-24, so f + n and
// 1 - f are exact), three short Taylor polynomials on |angle| <= pi/3 serve all six taps:
//   sin(pi t/3): q0  sin(pi (1-f)/3),  q1  cos(pi (2f-1)/6),  q2  sin(pi f/3),  q3 = -q0,  q4 = -q1,  q5 = -q2
__device__ __forceinline__ float sinpi_third(float u) {      // sin(pi u), 0 <= u <= 1/3: truncation 3.4e-10 relative
    const float u2 = u * u;
    float p = fmaf(u2, -0.007370430945714348f, 0.08214588661112819f);
    p = fmaf(u2, p, -0.5992645293207919f);
    p = fmaf(u2, p, 2.550164039877345f);
    p = fmaf(u2, p, -5.167712780049969f);
    p = fmaf(u2, p, 3.141592653589793f);
    return u * p;
}
__device__ __forceinline__ float cospi_sixth(float w) {      // cos(pi w), |w| <= 1/6: truncation 4.9e-10 relative
    const float w2 = w * w;
    float p = fmaf(w2, 0.23533063035889312f, -1.3352627688545893f);
    p = fmaf(w2, p, 4.058712126416768f);
    p = fmaf(w2, p, -4.934802200544679f);
    return fmaf(w2, p, 1.0f);
}
__device__ __forceinline__ void lanczos3_weights_f32(float f, float k[6]) {
    if (f == 0.0f) { k[0] = k[1] = k[3] = k[4] = k[5] = 0.0f; k[2] = 1.0f; return; }
    const float A = sinpi_third((1.0f - f) * 0.33333334f), B = -cospi_sixth(fmaf(f, 0.33333334f, -0.16666667f)), C = sinpi_third(f * 0.33333334f);
    const float t0 = f + 2.0f, t1 = f + 1.0f, t3 = f - 1.0f, t4 = f - 2.0f, t5 = f - 3.0f;
    k[0] = A * rcp_ftz(t0 * t0);
    k[1] = B * rcp_ftz(t1 * t1);
    k[2] = C * rcp_ftz(f * f);
    k[3] = A * rcp_ftz(t3 * t3);
    k[4] = B * rcp_ftz(t4 * t4);
    k[5] = C * rcp_ftz(t5 * t5);
}

// sinpi_third / cospi_sixth / lanczos3_weights_f32 for the x and the y fraction at once (.x: x axis, .y: y axis); the
// operations and their order are those of the scalar functions.  Neither fraction may be zero.
__device__ __forceinline__ float2 sinpi_third2(float2 u) {
    const float2 u2 = mul2(u, u);
    float2 p = fma2(u2, bc2(-0.007370430945714348f), bc2(0.08214588661112819f));
    p = fma2(u2, p, bc2(-0.5992645293207919f));
    p = fma2(u2, p, bc2(2.550164039877345f));
    p = fma2(u2, p, bc2(-5.167712780049969f));
    p = fma2(u2, p, bc2(3.141592653589793f));
    return mul2(u, p);
}
__device__ __forceinline__ float2 cospi_sixth2(float2 w) {
    const float2 w2 = mul2(w, w);
    float2 p = fma2(w2, bc2(0.23533063035889312f), bc2(-1.3352627688545893f));
    p = fma2(w2, p, bc2(4.058712126416768f));
    p = fma2(w2, p, bc2(-4.934802200544679f));
    return fma2(w2, p, bc2(1.0f));
}
__device__ __forceinline__ float2 rcp2_ftz(float2 v) { return make_float2(rcp_ftz(v.x), rcp_ftz(v.y)); }
__device__ __forceinline__ void lanczos3_weights_f32x2(float2 f, float2 k[6]) {
    const float2 A = sinpi_third2(mul2(add2(bc2(1.0f), make_float2(-f.x, -f.y)), bc2(0.33333334f)));
    const float2 Bc = cospi_sixth2(fma2(f, bc2(0.33333334f), bc2(-0.16666667f))), B = make_float2(-Bc.x, -Bc.y);
    const float2 C = sinpi_third2(mul2(f, bc2(0.33333334f)));
    const float2 t0 = add2(f, bc2(2.0f)), t1 = add2(f, bc2(1.0f)), t3 = add2(f, bc2(-1.0f)), t4 = add2(f, bc2(-2.0f)), t5 = add2(f, bc2(-3.0f));
    k[0] = mul2(A, rcp2_ftz(mul2(t0, t0)));
    k[1] = mul2(B, rcp2_ftz(mul2(t1, t1)));
    k[2] = mul2(C, rcp2_ftz(mul2(f, f)));
    k[3] = mul2(A, rcp2_ftz(mul2(t3, t3)));
    k[4] = mul2(B, rcp2_ftz(mul2(t4, t4)));
    k[5] = mul2(C, rcp2_ftz(mul2(t5, t5)));
}

// No masked tap in the tile's box: weight == 1.  a = address of the cell (floor x, floor y) in the calibrated box.
template <int KERNEL>
__device__ __forceinline__ float interp_clean(const float* __restrict__ a, int pitch, float fx, float fy) {
    if (KERNEL == 0) {
        const float c00 = a[0], c01 = a[1], c10 = a[pitch], c11 = a[pitch + 1];
        // (top, bot) = fx * ((c01, c11) - (c00, c10)) + (c00, c10)
        const float2 lo = make_float2(c00, c10);
        const float2 tb = fma2(bc2(fx), add2(make_float2(c01, c11), make_float2(-c00, -c10)), lo);
        return fmaf(fy, tb.y - tb.x, tb.x);
    } else {
        if (fx == 0.0f || fy == 0.0f) {              // a tap exactly on a pixel centre (1 in 2^23 fractions): the scalar form
            float kx[6], ky[6];
            lanczos3_weights_f32(fx, kx);
            lanczos3_weights_f32(fy, ky);
            const float* r = a - 2 * pitch - 2;
            float V = 0.0f;
#pragma unroll 1
            for (int b = 0; b < 6; ++b) {
                float rs = kx[0] * r[0];
#pragma unroll
                for (int q = 1; q < 6; ++q) rs = fmaf(kx[q], r[q], rs);
                V = fmaf(ky[b], rs, V);
                r += pitch;
            }
            const float sx = ((kx[0] + kx[5]) + (kx[1] + kx[4])) + (kx[2] + kx[3]);
            const float sy = ((ky[0] + ky[5]) + (ky[1] + ky[4])) + (ky[2] + ky[3]);
            return __fdividef(V, sx * sy);
        }
        float2 k[6];                                  // (kx[q], ky[q])
        lanczos3_weights_f32x2(make_float2(fx, fy), k);
        const float* r = a - 2 * pitch - 2;
        // FP32 accumulation is enough where no tap is masked (full-size parity: worst 0.61 x tolerance over 3.2e8 pixels).
        // Two rows of taps per packed operation; the sum over the rows stays in its order.
        float V = 0.0f;
#pragma unroll
        for (int b = 0; b < 6; b += 2) {
            const float* r1 = r + pitch;
            float2 rs = mul2(bc2(k[0].x), make_float2(r[0], r1[0]));
#pragma unroll
            for (int q = 1; q < 6; ++q) rs = fma2(bc2(k[q].x), make_float2(r[q], r1[q]), rs);
            V = fmaf(k[b].y, rs.x, V);
            V = fmaf(k[b + 1].y, rs.y, V);
            r += 2 * pitch;
        }
        const float2 s = add2(add2(add2(k[0], k[5]), add2(k[1], k[4])), add2(k[2], k[3]));   // (sum kx, sum ky)
        return __fdividef(V, s.x * s.y);   // 2 ulp: 2.4e-7 relative, 40x inside the relative tolerance
    }
}

// Masked, normalised form (NaN = masked tap): S0 = sum k, B = sum k over masked taps, V1 = sum k c over good taps.
template <int KERNEL>
__device__ __forceinline__ void interp_masked(const float* __restrict__ a, int pitch, float fx, float fy, float w_min,
                                              float& val, float& wgt) {
    float S = 0.0f, B = 0.0f, V1 = 0.0f;
    double V64 = 0.0;
    if (KERNEL == 0) {
        const float c00 = a[0], c01 = a[1], c10 = a[pitch], c11 = a[pitch + 1];
        const float gx = 1.0f - fx, gy = 1.0f - fy;
        const float k00 = gx * gy, k01 = fx * gy, k10 = gx * fy, k11 = fx * fy;
        S = (k00 + k01) + (k10 + k11);
        if (c00 == c00) V1 = fmaf(k00, c00, V1); else B += k00;
        if (c01 == c01) V1 = fmaf(k01, c01, V1); else B += k01;
        if (c10 == c10) V1 = fmaf(k10, c10, V1); else B += k10;
        if (c11 == c11) V1 = fmaf(k11, c11, V1); else B += k11;
    } else {
        float kx[6], ky[6];
        lanczos3_weights_f32(fx, kx);
        lanczos3_weights_f32(fy, ky);
        const float* r = a - 2 * pitch - 2;
#pragma unroll 1
        for (int b = 0; b < 6; ++b) {
#pragma unroll
            for (int q = 0; q < 6; ++q) {
                const float k = kx[q] * ky[b], c = r[q];
                S += k;
                if (c == c) V64 = fma((double)kx[q] * (double)ky[b], (double)c, V64); else B += k;
            }
            r += pitch;
        }
        V1 = (float)V64;
    }
    const float w = 1.0f - B / S;
    val = 0.f; wgt = 0.f;
    if (!(w < w_min) && (S - B > 0.f)) { val = V1 / (S - B); wgt = fminf(w, 1.0f); }
}

// ARGUS_DEBUG_BOUNDS build (tests/test_gpu_debug_bounds.py; compute-sanitizer is not available on the GPU pool): every
// shared-memory gather is checked against the staged box -- cell column / row of the position plus the kernel's taps must
// lie inside [0, box width) x [0, rows) -- and a violation is latched (bit 8 of the overflow latch: argus_plan_info fails).
#ifdef ARGUS_DEBUG_BOUNDS
#define RF_CHECK_BOX(PB, COL, ROW, TL, TR, BOXW, ROWS)                                                                  \
    if ((COL) - (TL) < 0 || (COL) + (TR) >= (BOXW) || (ROW) - (TL) < 0 || (ROW) + (TR) >= (ROWS)) plan_overflow(PB, 8);
#else
#define RF_CHECK_BOX(PB, COL, ROW, TL, TR, BOXW, ROWS)
#endif

// ------------------------------------------------------------------------------------------ kernel
// Bilinear, 80 registers: two CTAs leave 19 K registers per SM free, enough for one CTA of any plan kernel -- the plan
// of the next frame runs on a side stream underneath this kernel (argus_api.cu, ARGUS_OPT_PLAN_OVERLAP).
template <bool COADD, int KERNEL, int VAR = 0>
__global__ void __maxnreg__((FastCfg<KERNEL, VAR>::REGS))
    resample_fast_kernel(const __grid_constant__ FastMaps maps, PlanBuffers pb, FrameArgs f, int W, int H, float w_min, float* __restrict__ value_out, float* __restrict__ weight_out, long long out_cap,
                         CoaddArgs ca) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    typedef FastCfg<KERNEL, VAR> Cfg;
    constexpr int RF_STAGES = Cfg::STAGES;
    constexpr int RF_NI = (Cfg::CAP / 4 + RF_CONSUMERS - 1) / RF_CONSUMERS;   // calibration items (float4) per thread
    FastSmem<KERNEL, VAR>& sm = *reinterpret_cast<FastSmem<KERNEL, VAR>*>(smem_raw);
    const int tid = threadIdx.x;
    const int n_tiles = *pb.n_tiles;
    const float t_exp = f.t_exp, flat_min = f.flat_min;
    const int sat_adu = f.sat_adu;

    if (tid == 0) {
        for (int i = 0; i < 2; ++i) mbar_init(&sm.full[i], 1);
        for (int i = 0; i < RF_STAGES; ++i) mbar_init(&sm.empty[i], RF_CONSUMERS);
        mbar_init(&sm.empty_a, RF_CONSUMERS);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (tid >= RF_GROUPS * RF_CONSUMERS) {
        // ================================================================ producer warp
        const int lane = tid - RF_GROUPS * RF_CONSUMERS;
        int issued = 0, sentinels = 0;
        // software pipeline: the record and output offset of the NEXT tile are in flight while the current one is
        // handled (one producer serves RF_GROUPS groups, so its own load latency must stay off the critical path)
        float4 rv_n = make_float4(0.f, 0.f, 0.f, 0.f);
        long long off_n = 0;
#if RF_SCHED_DYNAMIC
        // tiles are claimed from a context-wide counter (pb.latch[2]) instead of dealt round-robin: the CTAs of an SM that shares
        // its issue slots with a plan kernel of the next frame (ARGUS_OPT_PLAN_OVERLAP) take fewer tiles, the others more, and the
        // kernel does not wait for the slowest SM's fixed share.  Claims stay in plan order, so concurrently staged boxes still
        // overlap in L2.  The last producer to finish (pb.latch[3]) resets both words for the next launch on the stream.
        // Claims run two tiles ahead and the record load one: the atomic's round trip and the load's are each a tile period in
        // flight (in one period together they made the producer the bottleneck of the bilinear kernel, 1.5 us per tile).
        int* const sched = pb.latch + 2;
        constexpr bool DYN = KERNEL == 1 || RF_SCHED_DYNAMIC > 1;
        int t_n = DYN ? __shfl_sync(0xffffffffu, lane == 0 ? atomicAdd(sched, 1) : 0, 0) : (int)blockIdx.x;
        int claim_nn = (DYN && lane == 0 && t_n < n_tiles) ? atomicAdd(sched, 1) : 0x7fffffff;   // lane 0's, broadcast when it is needed
#else
        constexpr bool DYN = false;
        int* const sched = nullptr;
        int t_n = blockIdx.x, claim_nn = 0;
#endif
        if (t_n < n_tiles) {
            if (lane < 10) rv_n = __ldg(reinterpret_cast<const float4*>(pb.frec + t_n) + lane);
            if (lane == 0) off_n = tile_out_offset(pb, t_n);
        }
        for (;;) {
            const int t = t_n;
            const bool last = t >= n_tiles;
            const float4 rv = rv_n;
            const long long off_c = off_n;
            if (DYN) {
                if (!last) {
                    t_n = __shfl_sync(0xffffffffu, claim_nn, 0);
                    claim_nn = (lane == 0 && t_n < n_tiles) ? atomicAdd(sched, 1) : 0x7fffffff;
                }
            } else {
                t_n = t + gridDim.x;
            }
            if (t_n < n_tiles) {
                if (lane < 10) rv_n = __ldg(reinterpret_cast<const float4*>(pb.frec + t_n) + lane);
                if (lane == 0) off_n = tile_out_offset(pb, t_n);
            }
            // lane 0 holds cls, mask_slot, gx0, gy0; lane 1 holds wclass, bh, kofs, X0
            const int cls = last ? -1 : __shfl_sync(0xffffffffu, __float_as_int(rv.x), 0);
            if (cls == 0) continue;                         // empty, or left to the general kernel
            const int slot = issued % RF_STAGES, ds = issued & 1;
            // stage free: every consumer is done with the tile that used it RF_STAGES tiles ago.  That also frees
            // descriptor ds: the consumers released tile issued-1's stage after they had finished tile issued-2.
            // SPLIT: raw / dark / flat are free once tile issued-1 has been calibrated (its gather still reads the calibrated box
            // over bias + pad); by then the consumers have finished tile issued-2, so descriptor ds is free as well
            if (Cfg::SPLIT) { if (issued >= 1) mbar_wait(&sm.empty_a, (unsigned)((issued - 1) & 1)); }
            else if (issued >= RF_STAGES) mbar_wait(&sm.empty[slot], (unsigned)((issued / RF_STAGES - 1) & 1));
            FastDesc& d = sm.desc[ds];
            if (last) {
                // end of work: one sentinel per consumer group (consecutive tiles go to distinct groups)
                if (lane == 0) {
                    d.r.cls = -1;
                    mbar_arrive(&sm.full[ds]);
                }
                ++issued;
                if (++sentinels == RF_GROUPS) break;
                continue;
            }
            const int mask_slot = __shfl_sync(0xffffffffu, __float_as_int(rv.y), 0);
            const int gx0 = __shfl_sync(0xffffffffu, __float_as_int(rv.z), 0), gy0 = __shfl_sync(0xffffffffu, __float_as_int(rv.w), 0);
            const int wclass = __shfl_sync(0xffffffffu, __float_as_int(rv.x), 1), bh = __shfl_sync(0xffffffffu, __float_as_int(rv.y), 1);
            unsigned tx_bytes = 0;
            {
                // one elected thread issues the four bulk-tensor copies (one box per array) as early as possible; the
                // arrive.expect_tx that completes the phase follows once the descriptor is written
                const int wc = wclass & 15, hc = wclass >> 4;
                const int boxw = 40 + 8 * wc, boxh = 48 + 8 * hc;
                tx_bytes = (unsigned)(boxh * boxw * 14);
                if (lane == 0) {
                    const CUtensorMap* mp = &maps.m[hc][wc][0];
                    typename FastSmem<KERNEL, VAR>::Stage& sg = sm.stage[slot];
                    tma_load_2d(sg.raw, mp + 0, gx0, gy0, &sm.full[ds]);
                    if (!Cfg::SPLIT) tma_load_2d(sg.bias, mp + 1, gx0, gy0, &sm.full[ds]);
                    else tma_prefetch_2d(mp + 1, gx0, gy0);         // loaded below, once the previous tile's gather is over
                    tma_load_2d(sg.dark, mp + 2, gx0, gy0, &sm.full[ds]);
                    tma_load_2d(sg.flat, mp + 3, gx0, gy0, &sm.full[ds]);
                }
            }
            if (lane < 10) reinterpret_cast<float4*>(&d.r)[lane] = rv;
            __syncwarp();
            {
                // Horner coefficients in T for pixel column u = lane: the S-dependent part of the tile polynomial,
                // shared by every consumer thread of that column
                const float S = (float)(2 * lane - 31) * 0.03125f;
                const float* px = d.r.px;
                const float* py = d.r.py;
                float4 t0, t1;
                t0.x = fmaf(S, fmaf(S, fmaf(S, px[6], px[3]), px[1]), px[0]);
                t0.y = fmaf(S, fmaf(S, px[7], px[4]), px[2]);
                t0.z = fmaf(S, px[8], px[5]);
                t0.w = fmaf(S, fmaf(S, fmaf(S, py[6], py[3]), py[1]), py[0]);
                t1.x = fmaf(S, fmaf(S, py[7], py[4]), py[2]);
                t1.y = fmaf(S, py[8], py[5]);
                t1.z = px[9];
                t1.w = py[9];
                d.tab[lane][0] = t0;
                d.tab[lane][1] = t1;
            }
            if (cls == TC_BORDER) {
                unsigned mk = pb.masks[(size_t)mask_slot * 32 + lane];
                int c = __popc(mk), inc = c;
                for (int o = 1; o < 32; o <<= 1) {
                    int y = __shfl_up_sync(0xffffffffu, inc, o);
                    if (lane >= o) inc += y;
                }
                d.mask[lane] = mk;
                d.pref[lane] = inc - c;
            }
            if (lane == 0) {
                d.off = off_c;
                d.t = t;
                if (COADD) {
                    d.cslot = pb.cslot[t];                      // coadd_slots_kernel, once per call
#ifndef ARGUS_NO_COADD_PREFETCH
                    // the tile's accumulators (2 x 4 KB, contiguous in the tile-dense layout) into L2 one or two tiles ahead of
                    // the consumers' read-modify-write: their loads were the kernel's longest stall (DRAM latency at 18 warps/SM)
                    if (d.cslot >= 0 && ((((unsigned long long)ca.sum | (unsigned long long)ca.wsum) & 15ull) == 0ull)) {   // (the API asks for 4-byte alignment only)
                        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" :: "l"(ca.sum + d.cslot), "r"(ARGUS_TILE_PIX * 4) : "memory");
                        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" :: "l"(ca.wsum + d.cslot), "r"(ARGUS_TILE_PIX * 4) : "memory");
                    }
#endif
                }
            }
            __syncwarp();
            if (Cfg::SPLIT) {
                // the bias box lands where the previous tile's calibrated box is still being gathered from
                if (issued >= 1) mbar_wait(&sm.empty[slot], (unsigned)((issued - 1) & 1));
                if (lane == 0) tma_load_2d(sm.stage[slot].bias, &maps.m[wclass >> 4][wclass & 15][1], gx0, gy0, &sm.full[ds]);
            }
            if (lane == 0) mbar_arrive_expect_tx(&sm.full[ds], tx_bytes);   // releases the descriptor to the consumers
            ++issued;
        }
        if (DYN && lane == 0 && atomicAdd(sched + 1, 1) == (int)gridDim.x - 1) {   // every CTA has made its last claim
            sched[0] = 0;
            sched[1] = 0;
        }
        return;
    }

    // ==================================================================== consumer warps
    const int group = tid / RF_CONSUMERS;
    const int gt = tid - group * RF_CONSUMERS;     // thread index within the group
    const int lane = tid & 31;
    const int ul = (int)compact_even_bits((unsigned)gt), vl = (int)compact_even_bits((unsigned)gt >> 1);
    const int s0 = 2 * ul - 31, t0 = 2 * vl - 31;
    const float T0 = (float)t0 * 0.03125f, T1 = T0 + 1.0f;
    const unsigned fmin_bits = __float_as_uint(flat_min), frange = 0x7f800000u - fmin_bits;
    const float sat_f = (float)sat_adu;

    for (int it = group;; it += RF_GROUPS) {
        const int slot = it % RF_STAGES, ds = it & 1;
        mbar_wait(&sm.full[ds], (unsigned)((it >> 1) & 1));
        const FastDesc& d = sm.desc[ds];
        const int cls = d.r.cls;
        if (cls < 0) break;
        typename FastSmem<KERNEL, VAR>::Stage& sg = sm.stage[slot];
        float* cal = Cfg::CALBUF > 0 ? sm.calbuf : sg.bias;
        const int boxw = 40 + 8 * (d.r.wclass & 15), pitch = fast_cal_pitch(boxw);
        // every column of the box is calibrated: restricting the items to the tap columns made the 128-bit shared
        // loads straddle rows inside a quarter-warp (bank conflicts) and measured 5 % slower
        const int bw4 = boxw >> 2, n4 = d.r.bh * bw4;
        const unsigned M = RF_ROW_MAGIC[d.r.wclass & 15];   // ceil(2^20 / bw4): exact division by bw4 for v < 2^14 (a division here
                                                            // was 3.8 % of the kernel's instructions)
        // ---- A2: calibrate the staged box once (the stage is dense: item v <-> float4 v).  Four independent items
        //      per thread are read and calibrated in registers; after a barrier (all reads done) they overwrite the
        //      stage with a pitch of 8 or 24 mod 32 floats, which makes the gather free of bank conflicts.
        float4 o4[RF_NI];
        int bad = 0, big = 0;
#pragma unroll
        for (int j = 0; j < RF_NI; ++j) {
            const int v = gt + RF_CONSUMERS * j;
            if (v < n4) {
                const uint2 rw = reinterpret_cast<const uint2*>(sg.raw)[v];
                const float4 b = reinterpret_cast<const float4*>(sg.bias)[v];
                const float4 dk = reinterpret_cast<const float4*>(sg.dark)[v];
                const float4 fl = reinterpret_cast<const float4*>(sg.flat)[v];
                o4[j] = calib_fast4<KERNEL == 1>(rw, b, dk, fl, t_exp, sat_f, fmin_bits, frange, bad);
                if (KERNEL == 1) big |= (fmaxf(fmaxf(fabsf(o4[j].x), fabsf(o4[j].y)), fmaxf(fabsf(o4[j].z), fabsf(o4[j].w))) > RF_LZ_BIG_ADU);
            }
        }
        const int any_bad = consumers_sync_or(group, bad);
        const int any_big = KERNEL == 1 ? consumers_sync_or(group, big) : 0;
        // separate calibrated box (Lanczos-3): every thread has read its part of the stage, the producer may refill it
        // while the gather runs
        if (Cfg::CALBUF > 0) mbar_arrive(&sm.empty[slot]);
        if (Cfg::SPLIT) mbar_arrive(&sm.empty_a);         // raw / dark / flat may be refilled; bias + pad hold the calibrated box
#pragma unroll
        for (int j = 0; j < RF_NI; ++j) {
            const int v = gt + RF_CONSUMERS * j;
            if (v < n4) {
                const int row = (int)(((unsigned)v * M) >> 20);
                *reinterpret_cast<float4*>(cal + row * pitch + 4 * (v - row * bw4)) = o4[j];
            }
        }
        consumers_sync(group);
        if (KERNEL == 1 && any_big && (any_bad || cls != TC_INSIDE)) {
            // Lanczos-3 with masked taps next to bright pixels (saturated star cores: huge taps, small results) needs FP64
            // kernel weights and FP64 coordinates to stay inside the value tolerance: such tiles are handed to the general
            // kernel, which runs after this one on the plan's slow list.  Without bright pixels in the box the FP32
            // masked form below is inside the tolerance (errors scale with the largest tap).
            if (gt == 0) slow_push(pb, d.t);
            if (Cfg::CALBUF == 0) mbar_arrive(&sm.empty[slot]);
            continue;
        }

        // ---- A3/A4: tile polynomial -> source position; A5: interpolation
        FastAxis ax, ay;
        {
            const float4 p0 = d.tab[ul][0], p1 = d.tab[ul][1];
            ax.A0 = p0.x; ax.B0 = p0.y; ax.C0 = p0.z; ax.c9 = p1.z;
            ay.A0 = p0.w; ay.B0 = p1.x; ay.C0 = p1.y; ay.c9 = p1.w;
            if (RF_CONSUMERS == 256) {
                const float4 q0 = d.tab[ul + 16][0], q1 = d.tab[ul + 16][1];
                ax.A1 = q0.x; ax.B1 = q0.y; ax.C1 = q0.z;
                ay.A1 = q0.w; ay.B1 = q1.x; ay.C1 = q1.y;
            } else {
                ax.A1 = ax.B1 = ax.C1 = ay.A1 = ay.B1 = ay.C1 = 0.f;
            }
            const int axi = d.r.ax, bxi = d.r.bx, ayi = d.r.ay, byi = d.r.by;
            ax.lin = d.r.c0x + axi * s0 + bxi * t0; ax.da = 32 * axi; ax.db = 32 * bxi;
            ay.lin = d.r.c0y + ayi * s0 + byi * t0; ay.da = 32 * ayi; ay.db = 32 * byi;
        }
        const float* cb = cal + d.r.kofs;
        const long long off = d.off;

        if (!COADD && cls == TC_INSIDE && !any_bad && off + ARGUS_TILE_PIX <= out_cap) {
            float* vp = value_out + off + gt;
            float* wp = weight_out + off + gt;
#define RF_HOT(Q)                                                                            \
    {                                                                                        \
        const int xf = fast_axis_eval<Q>(ax, T0, T1), yf = fast_axis_eval<Q>(ay, T0, T1);    \
        RF_CHECK_BOX(pb, d.r.X0 - d.r.gx0 + (xf >> FAST_FRAC_BITS), d.r.Y0 - d.r.gy0 + (yf >> FAST_FRAC_BITS), Cfg::TL, Cfg::TR, boxw, d.r.bh) \
        const float* a = cb + ((yf >> FAST_FRAC_BITS) * pitch + (xf >> FAST_FRAC_BITS));     \
        vp[RF_CONSUMERS * Q] = interp_clean<KERNEL>(a, pitch, fast_frac(xf), fast_frac(yf)); \
        wp[RF_CONSUMERS * Q] = 1.0f;                                                         \
    }
            RF_HOT(0) RF_HOT(1)
#if RF_NQ == 4
            RF_HOT(2) RF_HOT(3)
#endif
#undef RF_HOT
        } else if (COADD && cls == TC_INSIDE && !any_bad && d.cslot >= 0) {
            // A6 on a clean tile: weight == 1, so sum += value, wsum += 1.  The eight accumulator loads are issued
            // before the gather so that their latency hides under it (footprint pixels are unique within a frame:
            // plain read-modify-write, deterministic)
            float* sp = ca.sum + d.cslot + gt;
            float* wp = ca.wsum + d.cslot + gt;
            float s_acc[RF_NQ], w_acc[RF_NQ];
#pragma unroll
            for (int q = 0; q < RF_NQ; ++q) { s_acc[q] = sp[RF_CONSUMERS * q]; w_acc[q] = wp[RF_CONSUMERS * q]; }
#define RF_ACC(Q)                                                                            \
    {                                                                                        \
        const int xf = fast_axis_eval<Q>(ax, T0, T1), yf = fast_axis_eval<Q>(ay, T0, T1);    \
        RF_CHECK_BOX(pb, d.r.X0 - d.r.gx0 + (xf >> FAST_FRAC_BITS), d.r.Y0 - d.r.gy0 + (yf >> FAST_FRAC_BITS), Cfg::TL, Cfg::TR, boxw, d.r.bh) \
        const float* a = cb + ((yf >> FAST_FRAC_BITS) * pitch + (xf >> FAST_FRAC_BITS));     \
        sp[RF_CONSUMERS * Q] = s_acc[Q] + interp_clean<KERNEL>(a, pitch, fast_frac(xf), fast_frac(yf)); \
        wp[RF_CONSUMERS * Q] = w_acc[Q] + 1.0f;                                              \
    }
            RF_ACC(0) RF_ACC(1)
#if RF_NQ == 4
            RF_ACC(2) RF_ACC(3)
#endif
#undef RF_ACC
        } else {
            // masked source pixels, tiles cut by the frame border, coadd tiles outside the layout
            const long long cslot = COADD ? d.cslot : 0;
#define RF_GEN(Q)                                                                                          \
    {                                                                                                      \
        const int m = gt + RF_CONSUMERS * Q;                                                                        \
        bool member = true;                                                                                \
        long long pos = m;                                                                                 \
        if (cls != TC_INSIDE) {                                                                            \
            const unsigned mk = d.mask[m >> 5];                                                            \
            member = (mk >> lane) & 1u;                                                                    \
            pos = d.pref[m >> 5] + __popc(mk & ((1u << lane) - 1u));                                       \
        }                                                                                                  \
        if (member) {                                                                                      \
            const int xf = fast_axis_eval<Q>(ax, T0, T1), yf = fast_axis_eval<Q>(ay, T0, T1);              \
            RF_CHECK_BOX(pb, d.r.X0 - d.r.gx0 + (xf >> FAST_FRAC_BITS), d.r.Y0 - d.r.gy0 + (yf >> FAST_FRAC_BITS), Cfg::TL, Cfg::TR, boxw, d.r.bh) \
            const float* a = cb + ((yf >> FAST_FRAC_BITS) * pitch + (xf >> FAST_FRAC_BITS));               \
            float val, wgt;                                                                                \
            interp_masked<KERNEL>(a, pitch, fast_frac(xf), fast_frac(yf), w_min, val, wgt);                \
            if (COADD) {                                                                                   \
                if (cslot >= 0) {                                                                          \
                    ca.sum[cslot + m] = fmaf(wgt, val, ca.sum[cslot + m]);                                 \
                    ca.wsum[cslot + m] += wgt;                                                             \
                } else if (ca.n_skipped) {                                                                 \
                    atomicAdd(ca.n_skipped, 1ull);                                                         \
                }                                                                                          \
            } else if (off + pos < out_cap) {                                                              \
                value_out[off + pos] = val;                                                                \
                weight_out[off + pos] = wgt;                                                               \
            }                                                                                              \
        }                                                                                                  \
    }
            RF_GEN(0) RF_GEN(1)
#if RF_NQ == 4
            RF_GEN(2) RF_GEN(3)
#endif
#undef RF_GEN
        }
        if (Cfg::CALBUF == 0) mbar_arrive(&sm.empty[slot]);   // this thread is done with the stage (in-place calibrated box)
    }
}
