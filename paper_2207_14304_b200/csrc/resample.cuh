// resample.cuh -- A2..A6 fused: calibrate-on-stage + HEALPix resampling (+ optional coadd accumulate).
//
// One CTA (256 threads) per 32x32 output tile (1024 consecutive nested indices), persistent loop:
//   1. stage   the source bounding box of the tile is read with coalesced 128-bit loads (raw uint16 x4,
//              masters float4), calibrated ONCE in registers and stored to shared memory
//              as float32 (masked pixels as NaN); the calibrated frame never exists in HBM;
//   2. gather  each thread evaluates the tile-local coordinates of 4 output pixels (Morton index
//              tid + 256 q, so that every store instruction of a warp writes 32 consecutive floats),
//              gathers its taps from shared memory, interpolates and writes value and
//              weight -- or accumulates them into the coadd buffer.
// Tiles whose box has no masked pixel take a branch-free fast path (weight == 1).
#pragma once
#include <cuda_fp16.h>

#include "common.cuh"
#include "plan.cuh"

#define RS_THREADS 256
#define RS_BOX_FLOATS 6144   // shared-memory capacity of the staged source box (24 KB)
#define RS_MIN_CTAS 4         // register cap 64/thread -> 4 CTAs (32 warps) per SM

struct FrameArgs {
    const unsigned short* raw;
    const float* bias;
    const float* dark;
    const float* flat;
    const unsigned char* bpm;
    const float* cal;
    const unsigned char* mask;
    float t_exp, flat_min;
    int sat_adu;
    int vec_ok;   // W % 4 == 0 and all base pointers 16-byte aligned
    // pre-fused masters (argus_prepare_masters): offset = bias + dark * t_exp, gain = 1 / flat with NaN
    // where the pixel is invalid; float32 (pre = 1) or binary16 (pre = 2).  pre = 0: bias / dark / flat above.
    const void* offset;
    const void* gain;
    int pre;
};

struct CoaddArgs {
    const long long* tiles;
    long long n_tiles;
    int shift;            // layout tile id = plan tile id >> shift   (shift = 2 (k - k_tile) - 10)
    float* sum;
    float* wsum;
    unsigned long long* n_skipped;
};

__device__ __forceinline__ float nanf_() { return __int_as_float(0x7fc00000); }

// A2 for one pixel; masked -> NaN.
__device__ __forceinline__ float calib_px(float r, float b, float d, float fl, bool bad, float t_exp, float flat_min) {
    float t = fmaf(-d, t_exp, r - b);
    bool good = !bad && (fl >= flat_min) && (fl < INFINITY) && (fabsf(t) < INFINITY);
    return good ? __fdividef(t, fl) : nanf_();
}

// Lanczos-3 variant: the negative lobes cancel bright taps against each other, so the calibrated value is
// formed in FP64 and rounded once to float32 (0.5 ulp) -- DESIGN.md "Lanczos precision".
__device__ __forceinline__ float calib_px_precise(float r, float b, float d, float fl, bool bad, float t_exp, float flat_min) {
    double t = (double)r - (double)b - (double)d * (double)t_exp;
    bool good = !bad && (fl >= flat_min) && (fl < INFINITY) && (fabs(t) < (double)INFINITY);
    return good ? (float)(t / (double)fl) : nanf_();
}
template <bool PRECISE>
__device__ __forceinline__ float calib_sel(float r, float b, float d, float fl, bool bad, float t_exp, float flat_min) {
    return PRECISE ? calib_px_precise(r, b, d, fl, bad, t_exp, flat_min) : calib_px(r, b, d, fl, bad, t_exp, flat_min);
}

// A2 with pre-fused masters (R-M4): cal = (raw - offset) * gain; masked (NaN) where raw is saturated or the gain is NaN.
template <bool PRECISE>
__device__ __forceinline__ float calib_pre(float r, float off, float g, bool bad) {
    const float c = PRECISE ? (float)(((double)r - (double)off) * (double)g) : (r - off) * g;
    return (!bad && fabsf(c) < INFINITY) ? c : nanf_();
}
__device__ __forceinline__ float pre_load(const void* p, size_t o, int pre) {
    return pre == 1 ? reinterpret_cast<const float*>(p)[o] : __half2float(reinterpret_cast<const __half*>(p)[o]);
}
// four consecutive pixels at element offset o (16-byte / 8-byte aligned there)
__device__ __forceinline__ float4 pre_load4(const void* p, size_t o, int pre) {
    if (pre == 1) return __ldg(reinterpret_cast<const float4*>(reinterpret_cast<const float*>(p) + o));
    const uint2 h = __ldg(reinterpret_cast<const uint2*>(reinterpret_cast<const __half*>(p) + o));
    const float2 a = __half22float2(*reinterpret_cast<const __half2*>(&h.x)), b = __half22float2(*reinterpret_cast<const __half2*>(&h.y));
    return make_float4(a.x, a.y, b.x, b.y);
}
template <bool PRECISE>
__device__ __forceinline__ float4 calib4_pre(const FrameArgs& f, size_t o) {
    const uint2 rw = __ldg(reinterpret_cast<const uint2*>(f.raw + o));
    const float4 off = pre_load4(f.offset, o, f.pre), g = pre_load4(f.gain, o, f.pre);
    const int r0 = rw.x & 0xffff, r1 = rw.x >> 16, r2 = rw.y & 0xffff, r3 = rw.y >> 16;
    return make_float4(calib_pre<PRECISE>((float)r0, off.x, g.x, r0 >= f.sat_adu), calib_pre<PRECISE>((float)r1, off.y, g.y, r1 >= f.sat_adu),
                       calib_pre<PRECISE>((float)r2, off.z, g.z, r2 >= f.sat_adu), calib_pre<PRECISE>((float)r3, off.w, g.w, r3 >= f.sat_adu));
}

template <bool FUSED, bool PRECISE = false>
__device__ __forceinline__ float load_px(const FrameArgs& f, int W, int H, int gx, int gy) {
    if (gx < 0 || gx >= W || gy < 0 || gy >= H) return nanf_();
    size_t o = (size_t)gy * W + gx;
    if (FUSED && f.pre) {
        const int r = f.raw[o];
        return calib_pre<PRECISE>((float)r, pre_load(f.offset, o, f.pre), pre_load(f.gain, o, f.pre), r >= f.sat_adu);
    }
    if (FUSED) {
        int r = f.raw[o];
        bool bad = (r >= f.sat_adu) || (f.bpm && f.bpm[o] != 0);
        return calib_sel<PRECISE>((float)r, f.bias[o], f.dark[o], f.flat[o], bad, f.t_exp, f.flat_min);
    } else {
        return f.mask[o] ? f.cal[o] : nanf_();
    }
}

// A2 for one pixel on the fast (bilinear) path: raw arrives as a 16-bit field, converted with the
// 2^23 magic-number trick (exact), divided with rcp.approx.ftz (2 ulp: DESIGN.md "calibration precision");
// flat_min <= flat < +inf is one unsigned range compare on the float bits (flat_min > 0 enforced by the API).
__device__ __forceinline__ float rcp_ftz(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// REFINE: one Newton step on the quotient (<= 1 ulp) for the Lanczos-3 path, whose negative lobes amplify relative errors.
template <bool REFINE = false>
__device__ __forceinline__ float calib_fast(unsigned magic_r, float b, float d, float fl, bool bpm_bad, float t_exp,
                                            float sat_f, unsigned fmin_bits, unsigned frange) {
    float rf = __uint_as_float(magic_r) - 8388608.0f;
    const float t = fmaf(-d, t_exp, rf - b), r = rcp_ftz(fl);
    float c = t * r;
    if (REFINE) c = fmaf(fmaf(-c, fl, t), r, c);
    bool good = !bpm_bad && (rf < sat_f) && ((__float_as_uint(fl) - fmin_bits) < frange) && (fabsf(c) < INFINITY);
    return good ? c : nanf_();
}

// Four consecutive pixels through calib_fast, two per packed FP32 instruction (the operations and their order are
// calib_fast's: bit-identical).  rw: the four 16-bit raw values.
template <bool REFINE = false>
__device__ __forceinline__ float4 calib_fast4(uint2 rw, float4 b, float4 d, float4 fl, float t_exp, float sat_f, unsigned fmin_bits,
                                              unsigned frange, int& bad) {
    const float2 m01 = make_float2(__uint_as_float(__byte_perm(rw.x, 0x4B000000u, 0x7610)), __uint_as_float(__byte_perm(rw.x, 0x4B000000u, 0x7632)));
    const float2 m23 = make_float2(__uint_as_float(__byte_perm(rw.y, 0x4B000000u, 0x7610)), __uint_as_float(__byte_perm(rw.y, 0x4B000000u, 0x7632)));
    const float2 rf01 = add2(m01, bc2(-8388608.0f)), rf23 = add2(m23, bc2(-8388608.0f));
    const float2 t01 = fma2(make_float2(-d.x, -d.y), bc2(t_exp), add2(rf01, make_float2(-b.x, -b.y)));
    const float2 t23 = fma2(make_float2(-d.z, -d.w), bc2(t_exp), add2(rf23, make_float2(-b.z, -b.w)));
    const float2 r01 = make_float2(rcp_ftz(fl.x), rcp_ftz(fl.y)), r23 = make_float2(rcp_ftz(fl.z), rcp_ftz(fl.w));
    float2 c01 = mul2(t01, r01), c23 = mul2(t23, r23);
    if (REFINE) {
        c01 = fma2(fma2(make_float2(-c01.x, -c01.y), make_float2(fl.x, fl.y), t01), r01, c01);
        c23 = fma2(fma2(make_float2(-c23.x, -c23.y), make_float2(fl.z, fl.w), t23), r23, c23);
    }
    // all four good (the usual case) from three maxima: no per-pixel predicate logic and no selects on that path
    const float rmax = fmaxf(fmaxf(rf01.x, rf01.y), fmaxf(rf23.x, rf23.y));
    const unsigned fmax = max(max(__float_as_uint(fl.x) - fmin_bits, __float_as_uint(fl.y) - fmin_bits),
                              max(__float_as_uint(fl.z) - fmin_bits, __float_as_uint(fl.w) - fmin_bits));
    const float cmax = fmaxf(fmaxf(fabsf(c01.x), fabsf(c01.y)), fmaxf(fabsf(c23.x), fabsf(c23.y)));   // NaN operands drop out of fmaxf:
    const float2 cs2 = add2(c01, c23);
    const float csum = cs2.x + cs2.y;                                                                   // ... so NaN is caught by the sum
    if ((rmax < sat_f) && (fmax < frange) && (cmax < INFINITY) && (csum == csum)) return make_float4(c01.x, c01.y, c23.x, c23.y);
    const bool g0 = (rf01.x < sat_f) && ((__float_as_uint(fl.x) - fmin_bits) < frange) && (fabsf(c01.x) < INFINITY);
    const bool g1 = (rf01.y < sat_f) && ((__float_as_uint(fl.y) - fmin_bits) < frange) && (fabsf(c01.y) < INFINITY);
    const bool g2 = (rf23.x < sat_f) && ((__float_as_uint(fl.z) - fmin_bits) < frange) && (fabsf(c23.x) < INFINITY);
    const bool g3 = (rf23.y < sat_f) && ((__float_as_uint(fl.w) - fmin_bits) < frange) && (fabsf(c23.y) < INFINITY);
    bad |= !(g0 && g1 && g2 && g3);                  // a masked pixel among the four (the caller need not test for NaN)
    return make_float4(g0 ? c01.x : nanf_(), g1 ? c01.y : nanf_(), g2 ? c23.x : nanf_(), g3 ? c23.y : nanf_());
}

// Stage the box [gx0, gx0+bw) x [gy0, gy0+bh) (gx0, bw multiples of 4) into s_box (pitch bw).
// Returns non-zero for threads that stored a masked pixel.
template <bool FUSED, bool PRECISE>
__device__ __forceinline__ int stage_box(const FrameArgs& f, int W, int H, int gx0, int gy0, int bw, int bh,
                                         float* s_box, int tid) {
    int bad_any = 0;
    const int bw4 = bw >> 2, nvec = bw4 * bh;
    const unsigned M = (1048576u + bw4 - 1) / bw4;   // exact division by bw4 for v < 2^14
    const unsigned fmin_bits = __float_as_uint(f.flat_min), frange = 0x7f800000u - fmin_bits;
    const float sat_f = (float)f.sat_adu;
    for (int v = tid; v < nvec; v += RS_THREADS) {
        int row = (int)(((unsigned)v * M) >> 20);
        int c4 = v - row * bw4;
        int gy = gy0 + row, gx = gx0 + 4 * c4;
        float4 o4;
        if (f.vec_ok && (unsigned)gy < (unsigned)H && gx >= 0 && gx + 3 < W) {
            unsigned o = (unsigned)gy * (unsigned)W + (unsigned)gx;   // vec_ok implies W*H < 2^31
            if (FUSED && f.pre) {
                o4 = calib4_pre<PRECISE>(f, o);
            } else if (FUSED) {
                uint2 rw = __ldg(reinterpret_cast<const uint2*>(f.raw + o));
                float4 b = __ldg(reinterpret_cast<const float4*>(f.bias + o));
                float4 d = __ldg(reinterpret_cast<const float4*>(f.dark + o));
                float4 fl = __ldg(reinterpret_cast<const float4*>(f.flat + o));
                unsigned bp = 0;
                if (f.bpm) bp = __ldg(reinterpret_cast<const unsigned*>(f.bpm + o));
                if (PRECISE) {
                    int r0 = rw.x & 0xffff, r1 = rw.x >> 16, r2 = rw.y & 0xffff, r3 = rw.y >> 16;
                    o4.x = calib_px_precise((float)r0, b.x, d.x, fl.x, r0 >= f.sat_adu || (bp & 0xffu), f.t_exp, f.flat_min);
                    o4.y = calib_px_precise((float)r1, b.y, d.y, fl.y, r1 >= f.sat_adu || (bp & 0xff00u), f.t_exp, f.flat_min);
                    o4.z = calib_px_precise((float)r2, b.z, d.z, fl.z, r2 >= f.sat_adu || (bp & 0xff0000u), f.t_exp, f.flat_min);
                    o4.w = calib_px_precise((float)r3, b.w, d.w, fl.w, r3 >= f.sat_adu || (bp & 0xff000000u), f.t_exp, f.flat_min);
                } else {
                    o4.x = calib_fast(__byte_perm(rw.x, 0x4B000000u, 0x7610), b.x, d.x, fl.x, bp & 0xffu, f.t_exp, sat_f, fmin_bits, frange);
                    o4.y = calib_fast(__byte_perm(rw.x, 0x4B000000u, 0x7632), b.y, d.y, fl.y, bp & 0xff00u, f.t_exp, sat_f, fmin_bits, frange);
                    o4.z = calib_fast(__byte_perm(rw.y, 0x4B000000u, 0x7610), b.z, d.z, fl.z, bp & 0xff0000u, f.t_exp, sat_f, fmin_bits, frange);
                    o4.w = calib_fast(__byte_perm(rw.y, 0x4B000000u, 0x7632), b.w, d.w, fl.w, bp & 0xff000000u, f.t_exp, sat_f, fmin_bits, frange);
                }
            } else {
                float4 c = __ldg(reinterpret_cast<const float4*>(f.cal + o));
                unsigned mk = __ldg(reinterpret_cast<const unsigned*>(f.mask + o));
                o4.x = (mk & 0xffu) ? c.x : nanf_();
                o4.y = (mk & 0xff00u) ? c.y : nanf_();
                o4.z = (mk & 0xff0000u) ? c.z : nanf_();
                o4.w = (mk & 0xff000000u) ? c.w : nanf_();
            }
        } else {
            o4.x = load_px<FUSED, PRECISE>(f, W, H, gx, gy);
            o4.y = load_px<FUSED, PRECISE>(f, W, H, gx + 1, gy);
            o4.z = load_px<FUSED, PRECISE>(f, W, H, gx + 2, gy);
            o4.w = load_px<FUSED, PRECISE>(f, W, H, gx + 3, gy);
        }
        bad_any |= (o4.x != o4.x) | (o4.y != o4.y) | (o4.z != o4.z) | (o4.w != o4.w);
        *reinterpret_cast<float4*>(s_box + row * bw + 4 * c4) = o4;
    }
    return bad_any;
}

// Tap fetchers: shared-memory box, or (fallback for boxes that do not fit) straight from global memory.
struct SmemTaps {
    const float* s;
    int gx0, gy0, pitch;
    __device__ __forceinline__ float operator()(int i, int j) const { return s[(j - gy0) * pitch + (i - gx0)]; }
};
template <bool FUSED, bool PRECISE = false>
struct GlobalTaps {
    const FrameArgs* f;
    int W, H;
    __device__ __forceinline__ float operator()(int i, int j) const { return load_px<FUSED, PRECISE>(*f, W, H, i, j); }
};

// A5 masked, normalised bilinear (general path).
template <class Taps>
__device__ __forceinline__ void interp_bilinear_masked(const Taps& tp, int i, int j, float fx, float fy, float w_min,
                                                       float& val, float& wgt) {
    float c00 = tp(i, j), c01 = tp(i + 1, j), c10 = tp(i, j + 1), c11 = tp(i + 1, j + 1);
    float gx = 1.0f - fx, gy = 1.0f - fy;
    float k00 = gx * gy, k01 = fx * gy, k10 = gx * fy, k11 = fx * fy;
    float S0 = (k00 + k01) + (k10 + k11);
    float B = 0.f, V1 = 0.f;
    if (c00 == c00) V1 = fmaf(k00, c00, V1); else B += k00;
    if (c01 == c01) V1 = fmaf(k01, c01, V1); else B += k01;
    if (c10 == c10) V1 = fmaf(k10, c10, V1); else B += k10;
    if (c11 == c11) V1 = fmaf(k11, c11, V1); else B += k11;
    float w = 1.0f - B / S0;
    if (w < w_min || !(S0 - B > 0.f)) { val = 0.f; wgt = 0.f; }
    else { val = V1 / (S0 - B); wgt = fminf(w, 1.0f); }
}

// Lanczos-3 weights of the six taps i0-2 .. i0+3 for fraction f in [0,1), up to a common factor: L(t) = sinc(t)
// sinc(t/3) = sin(pi t) sin(pi t/3) 3 / (pi t)^2 and sin(pi t_q) = (-1)^q sin(pi f) for t_q = f + 2 - q, so the
// factor 3 sin(pi f) / pi^2 is shared by all six taps and cancels in value = V1 / (S0 - B) and in weight = 1 - B/S0.
// FP64 (general kernel: DESIGN.md "Lanczos precision"); three trigonometric evaluations serve the six taps:
//   sin(pi t/3): q0  sin(pi (1-f)/3),  q1  cos(pi (2f-1)/6),  q2  sin(pi f/3),  q3 = -q0,  q4 = -q1,  q5 = -q2
__device__ __forceinline__ void lanczos3_weights(double fd, double k[6]) {
    if (fd == 0.0) { k[0] = k[1] = k[3] = k[4] = k[5] = 0.0; k[2] = 1.0; return; }
    const double A = sinpi((1.0 - fd) * (1.0 / 3.0)), B = -cospi((2.0 * fd - 1.0) * (1.0 / 6.0)), C = sinpi(fd * (1.0 / 3.0));
    const double t0 = fd + 2.0, t1 = fd + 1.0, t3 = fd - 1.0, t4 = fd - 2.0, t5 = fd - 3.0;
    k[0] = A / (t0 * t0);
    k[1] = B / (t1 * t1);
    k[2] = C / (fd * fd);
    k[3] = A / (t3 * t3);
    k[4] = B / (t4 * t4);
    k[5] = C / (t5 * t5);
}

template <class Taps>
__device__ __forceinline__ void interp_lanczos3_masked(const Taps& tp, int i, int j, double fx, double fy, float w_min,
                                                       float& val, float& wgt) {
    double kx[6], ky[6];
    lanczos3_weights(fx, kx);
    lanczos3_weights(fy, ky);
    double S0 = 0.0, B = 0.0, V1 = 0.0;
#pragma unroll
    for (int b = 0; b < 6; ++b) {
#pragma unroll
        for (int a = 0; a < 6; ++a) {
            double k = kx[a] * ky[b];
            float c = tp(i - 2 + a, j - 2 + b);
            S0 += k;
            if (c == c) V1 = fma(k, (double)c, V1); else B += k;
        }
    }
    double w = 1.0 - B / S0;
    if (w < (double)w_min || !(S0 - B > 0.0)) { val = 0.f; wgt = 0.f; }
    else { val = (float)(V1 / (S0 - B)); wgt = (float)fmin(w, 1.0); }
}

// ------------------------------------------------------------------------------------------------
// The fused kernel.  KERNEL: 0 bilinear, 1 Lanczos-3.  FUSED: raw + masters (A2 fused) or cal + mask.
// COADD: accumulate into the coadd buffer instead of writing value / weight.
// ------------------------------------------------------------------------------------------------
template <int KERNEL, bool FUSED, bool COADD>
__global__ void __launch_bounds__(RS_THREADS, KERNEL == 0 ? RS_MIN_CTAS : 2) resample_tiles_kernel(DevWcs w, PlanBuffers pb, FrameArgs f, float w_min,
                                                                   float* __restrict__ value_out,
                                                                   float* __restrict__ weight_out, long long out_cap,
                                                                   CoaddArgs ca, int slow_only) {
    __shared__ __align__(16) float s_box[RS_BOX_FLOATS];
    __shared__ unsigned s_mask[32];
    __shared__ int s_pref[32];
    __shared__ long long s_slot;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int n_tiles = *pb.n_tiles;
    const int TL = KERNEL ? 2 : 0, TR = KERNEL ? 3 : 1;
    // this thread's pixels: Morton index m_q = tid + 256 q -> (u, v) = (ul + 16 (q & 1), vl + 16 (q >> 1))
    const int ul = (int)compact_even_bits((unsigned)tid), vl = (int)compact_even_bits((unsigned)tid >> 1);
    const int s0 = 2 * ul - 31, t0 = 2 * vl - 31;           // doubled centred offsets of pixel q = 0
    const float S0 = (float)s0 * 0.03125f, S1 = S0 + 1.0f, T0 = (float)t0 * 0.03125f, T1 = T0 + 1.0f;

    // slow_only: visit only the tiles the TMA-staged kernel (resample_fast.cuh) left to this one
    const int n_items = slow_only ? min(*pb.slow_count, pb.max_tiles) : n_tiles;
    for (int it = blockIdx.x; it < n_items; it += gridDim.x) {
        const int t = slow_only ? pb.slow_list[it] : it;
        const TileRec* __restrict__ rp = pb.rec + t;
        const int cls = rp->cls;
        if (cls == TC_EMPTY) continue;              // uniform over the CTA
        const long long off = tile_out_offset(pb, t);
        // source box (cells of floor(x), floor(y) plus the kernel's tap extent), x aligned to 4
        int gx0 = (rp->bx0 - TL) & ~3, gx1 = rp->bx1 + TR;
        int gy0 = rp->by0 - TL, gy1 = rp->by1 + TR;
        // clip to the frame plus the tap apron (everything beyond is off-frame = masked anyway)
        gx0 = max(gx0, -4); gx1 = min(gx1, w.W - 1 + TR); gy0 = max(gy0, -1 - TL); gy1 = min(gy1, w.H - 1 + TR);
        const int bw = ((gx1 - gx0 + 1) + 3) & ~3, bh = gy1 - gy0 + 1;
        const bool fits = (bw > 0 && bh > 0 && bw * bh <= RS_BOX_FLOATS);
        __syncthreads();                            // previous tile's gathers are done with s_box / s_mask
        int bad = 1;
        if (fits) bad = stage_box<FUSED, KERNEL == 1>(f, w.W, w.H, gx0, gy0, bw, bh, s_box, tid);
        if (cls != TC_INSIDE && wid == 0) {
            unsigned mk = pb.masks[(size_t)rp->mask_slot * 32 + lane];
            int c = __popc(mk), inc = c;
            for (int o = 1; o < 32; o <<= 1) {
                int y = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += y;
            }
            s_mask[lane] = mk;
            s_pref[lane] = inc - c;
        }
        if (COADD && tid == 0) {
            long long key = rp->tile >> ca.shift, lo = 0, hi = ca.n_tiles - 1, pos = -1;
            while (lo <= hi) {
                long long mid = (lo + hi) >> 1, tv = ca.tiles[mid];
                if (tv == key) { pos = mid; break; }
                if (tv < key) lo = mid + 1; else hi = mid - 1;
            }
            long long ppt = 1ll << (ca.shift + 10);
            s_slot = pos < 0 ? -1 : pos * ppt + ((rp->tile << 10) & (ppt - 1));
        }
        const int any_bad = __syncthreads_or(bad);

        if (KERNEL == 0 && !COADD && cls == TC_INSIDE && fits && !any_bad && off + ARGUS_TILE_PIX <= out_cap) {
            // ---- hot path: whole tile inside the frame, no masked source pixel, bilinear ----
            PolyAxis px, py;
            poly_axis_load(*rp, 0, px);
            poly_axis_load(*rp, 1, py);
            // Horner in T with S-dependent coefficients; pixels q and q^2 share S, q and q^1 share T
            float Ax0 = fmaf(S0, fmaf(S0, fmaf(S0, px.c6, px.c3), px.c1), px.c0), Ax1 = fmaf(S1, fmaf(S1, fmaf(S1, px.c6, px.c3), px.c1), px.c0);
            float Bx0 = fmaf(S0, fmaf(S0, px.c7, px.c4), px.c2), Bx1 = fmaf(S1, fmaf(S1, px.c7, px.c4), px.c2);
            float Cx0 = fmaf(S0, px.c8, px.c5), Cx1 = fmaf(S1, px.c8, px.c5);
            float Ay0 = fmaf(S0, fmaf(S0, fmaf(S0, py.c6, py.c3), py.c1), py.c0), Ay1 = fmaf(S1, fmaf(S1, fmaf(S1, py.c6, py.c3), py.c1), py.c0);
            float By0 = fmaf(S0, fmaf(S0, py.c7, py.c4), py.c2), By1 = fmaf(S1, fmaf(S1, py.c7, py.c4), py.c2);
            float Cy0 = fmaf(S0, py.c8, py.c5), Cy1 = fmaf(S1, py.c8, py.c5);
            const int hx00 = px.a * s0 + px.b * t0, hy00 = py.a * s0 + py.b * t0;
            const float* sb = s_box - (gy0 * bw + gx0);
            float* vp = value_out + off + tid;
            float* wp = weight_out + off + tid;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const float T = (q >> 1) ? T1 : T0;
                const float lox = fmaf(T, fmaf(T, fmaf(T, px.c9, (q & 1) ? Cx1 : Cx0), (q & 1) ? Bx1 : Bx0), (q & 1) ? Ax1 : Ax0);
                const float loy = fmaf(T, fmaf(T, fmaf(T, py.c9, (q & 1) ? Cy1 : Cy0), (q & 1) ? By1 : By0), (q & 1) ? Ay1 : Ay0);
                const int hx = hx00 + ((q & 1) ? 32 * px.a : 0) + ((q >> 1) ? 32 * px.b : 0);
                const int hy = hy00 + ((q & 1) ? 32 * py.a : 0) + ((q >> 1) ? 32 * py.b : 0);
                const float gxf = fmaf((float)(hx & 4095), 0.000244140625f, lox), gyf = fmaf((float)(hy & 4095), 0.000244140625f, loy);
                const float flx = floorf(gxf), fly = floorf(gyf);
                const float fx = gxf - flx, fy = gyf - fly;
                const int ci = px.base + (hx >> 12) + (int)flx, cj = py.base + (hy >> 12) + (int)fly;
                const float* a = sb + (cj * bw + ci);
                const float c00 = a[0], c01 = a[1], c10 = a[bw], c11 = a[bw + 1];
                const float top = fmaf(fx, c01 - c00, c00), bot = fmaf(fx, c11 - c10, c10);
                vp[256 * q] = fmaf(fy, bot - top, top);
                wp[256 * q] = 1.0f;
            }
            continue;
        }

        // ---- general path: border / exact tiles, masked pixels, Lanczos-3, coadd, oversized boxes ----
        PolyAxis px, py;
        int face = 0, ix0 = 0, iy0 = 0;
        if (cls == TC_EXACT) {
            int tx, ty;
            nest_to_xyf(rp->tile, w.k - ARGUS_TILE_LOG2, face, tx, ty);
            ix0 = tx * 32; iy0 = ty * 32;
        } else {
            poly_axis_load(*rp, 0, px);
            poly_axis_load(*rp, 1, py);
        }
        SmemTaps st{s_box, gx0, gy0, bw};
        GlobalTaps<FUSED, KERNEL == 1> gt{&f, w.W, w.H};
        const double* dc = pb.dcoef + (size_t)t * 20;
#pragma unroll 1
        for (int q = 0; q < 4; ++q) {
            const int m = tid + 256 * q;
            const int u = ul + 16 * (q & 1), v = vl + 16 * (q >> 1);
            long long pos = m;
            if (cls != TC_INSIDE) {
                unsigned mk = s_mask[m >> 5];
                if (!((mk >> lane) & 1u)) continue;
                pos = s_pref[m >> 5] + __popc(mk & ((1u << lane) - 1u));
            }
            int ci, cj;
            float fx, fy;
            double dfx = 0.0, dfy = 0.0;   // Lanczos-3 carries the fractions in FP64
            if (cls == TC_EXACT) {
                double x, y;
                pixel_to_xy(w, face, ix0 + u, iy0 + v, x, y);
                double flx = floor(x), fly = floor(y);
                ci = (int)flx; cj = (int)fly;
                dfx = x - flx; dfy = y - fly;
                fx = (float)dfx; fy = (float)dfy;
            } else if (KERNEL == 1) {
                poly_axis_eval_f64(dc, px, 2 * u - 31, 2 * v - 31, ci, dfx);
                poly_axis_eval_f64(dc + 10, py, 2 * u - 31, 2 * v - 31, cj, dfy);
                fx = (float)dfx; fy = (float)dfy;
            } else {
                poly_axis_eval(px, 2 * u - 31, 2 * v - 31, ci, fx);
                poly_axis_eval(py, 2 * u - 31, 2 * v - 31, cj, fy);
            }
            float val, wgt;
            if (fits) {
                // defensive clamp: the box covers every member pixel's taps by construction
                ci = min(max(ci, gx0 + TL), gx0 + bw - 1 - TR);
                cj = min(max(cj, gy0 + TL), gy0 + bh - 1 - TR);
                if (KERNEL == 0) interp_bilinear_masked(st, ci, cj, fx, fy, w_min, val, wgt);
                else interp_lanczos3_masked(st, ci, cj, dfx, dfy, w_min, val, wgt);
            } else {
                if (KERNEL == 0) interp_bilinear_masked(gt, ci, cj, fx, fy, w_min, val, wgt);
                else interp_lanczos3_masked(gt, ci, cj, dfx, dfy, w_min, val, wgt);
            }
            if (COADD) {
                long long sb = s_slot;
                if (sb >= 0) {
                    // footprint pixels are unique within a frame: plain read-modify-write, deterministic
                    ca.sum[sb + m] = fmaf(wgt, val, ca.sum[sb + m]);
                    ca.wsum[sb + m] += wgt;
                } else if (ca.n_skipped) {
                    atomicAdd(ca.n_skipped, 1ull);
                }
            } else {
                long long o = off + pos;
                if (o < out_cap) {
                    value_out[o] = val;
                    weight_out[o] = wgt;
                }
            }
        }
    }
    if (slow_only) {
        // The Lanczos-3 fast kernel appended run-time entries behind the plan's own (slow_plan).  The last CTA to finish
        // restores the list to the plan's state, so that a cached plan serves the next frame unchanged (no duplicates:
        // the coadd accumulation is not idempotent).  Every CTA read slow_count before it takes a ticket.
        __syncthreads();
        if (tid == 0) {
            __threadfence();
            if (atomicAdd(pb.ticket, 1u) == gridDim.x - 1) {
                *pb.slow_count = *pb.slow_plan;
                __threadfence();
                *pb.ticket = 0u;
            }
        }
    }
}

// Coadd slot of every plan tile for this call's layout, once per call (a binary search per tile in the producers of the
// staged kernels would sit on their critical path: 8 dependent loads per tile).
__global__ void __launch_bounds__(256) coadd_slots_kernel(PlanBuffers pb, CoaddArgs ca) {
    const int n = *pb.n_tiles;
    for (int t = blockIdx.x * 256 + threadIdx.x; t < n; t += gridDim.x * 256) {
        const long long tile = pb.tile_id[t];
        long long key = tile >> ca.shift, lo = 0, hi = ca.n_tiles - 1, pos = -1;
        while (lo <= hi) {
            const long long mid = (lo + hi) >> 1, tv = __ldg(ca.tiles + mid);
            if (tv == key) { pos = mid; break; }
            if (tv < key) lo = mid + 1; else hi = mid - 1;
        }
        const long long ppt = 1ll << (ca.shift + 10);
        pb.cslot[t] = pos < 0 ? -1 : pos * ppt + ((tile << 10) & (ppt - 1));
    }
}

// ------------------------------------------------------------------------------------------------
// General path for an explicit pixel list (argus_resample with idx != NULL): one thread per pixel,
// exact FP64 coordinates, taps straight from global memory.
// ------------------------------------------------------------------------------------------------
template <int KERNEL, bool FUSED>
__global__ void __launch_bounds__(256) resample_list_kernel(DevWcs w, FrameArgs f, float w_min,
                                                           const long long* __restrict__ idx, long long n,
                                                           float* __restrict__ value_out,
                                                           float* __restrict__ weight_out) {
    long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    long long p = idx[i];
    float val = 0.f, wgt = 0.f;
    long long npix = 12ll << (2 * w.k);
    if (p >= 0 && p < npix) {
        int face, ix, iy;
        nest_to_xyf(p, w.k, face, ix, iy);
        double x, y;
        double cosc = pixel_to_xy(w, face, ix, iy, x, y);
        if (cosc > 0.0 && fabs(x) < 1e9 && fabs(y) < 1e9) {
            double flx = floor(x), fly = floor(y);
            GlobalTaps<FUSED, KERNEL == 1> gt{&f, w.W, w.H};
            if (KERNEL == 0) interp_bilinear_masked(gt, (int)flx, (int)fly, (float)(x - flx), (float)(y - fly), w_min, val, wgt);
            else interp_lanczos3_masked(gt, (int)flx, (int)fly, x - flx, y - fly, w_min, val, wgt);
        }
    }
    value_out[i] = val;
    weight_out[i] = wgt;
}

// ------------------------------------------------------------------------------------------------
// A2 standalone: purely HBM-bound, 14 B in + 5 B out per pixel.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) calibrate_kernel(FrameArgs f, long long n, float* __restrict__ cal_out,
                                                       unsigned char* __restrict__ mask_out) {
    long long stride = (long long)gridDim.x * 256;
    if (f.vec_ok) {
        long long n4 = n >> 2;
        for (long long v = (long long)blockIdx.x * 256 + threadIdx.x; v < n4; v += stride) {
            size_t o = (size_t)v * 4;
            float c0, c1, c2, c3;
            if (f.pre) {
                const float4 c4 = calib4_pre<false>(f, o);
                c0 = c4.x; c1 = c4.y; c2 = c4.z; c3 = c4.w;
            } else {
                uint2 rw = __ldg(reinterpret_cast<const uint2*>(f.raw + o));
                float4 b = __ldg(reinterpret_cast<const float4*>(f.bias + o));
                float4 d = __ldg(reinterpret_cast<const float4*>(f.dark + o));
                float4 fl = __ldg(reinterpret_cast<const float4*>(f.flat + o));
                unsigned bp = f.bpm ? __ldg(reinterpret_cast<const unsigned*>(f.bpm + o)) : 0u;
                int r0 = rw.x & 0xffff, r1 = rw.x >> 16, r2 = rw.y & 0xffff, r3 = rw.y >> 16;
                c0 = calib_px((float)r0, b.x, d.x, fl.x, r0 >= f.sat_adu || (bp & 0xffu), f.t_exp, f.flat_min);
                c1 = calib_px((float)r1, b.y, d.y, fl.y, r1 >= f.sat_adu || (bp & 0xff00u), f.t_exp, f.flat_min);
                c2 = calib_px((float)r2, b.z, d.z, fl.z, r2 >= f.sat_adu || (bp & 0xff0000u), f.t_exp, f.flat_min);
                c3 = calib_px((float)r3, b.w, d.w, fl.w, r3 >= f.sat_adu || (bp & 0xff000000u), f.t_exp, f.flat_min);
            }
            unsigned mk = (c0 == c0 ? 1u : 0u) | (c1 == c1 ? 0x100u : 0u) | (c2 == c2 ? 0x10000u : 0u) | (c3 == c3 ? 0x1000000u : 0u);
            float4 o4 = make_float4(c0 == c0 ? c0 : 0.f, c1 == c1 ? c1 : 0.f, c2 == c2 ? c2 : 0.f, c3 == c3 ? c3 : 0.f);
            *reinterpret_cast<float4*>(cal_out + o) = o4;
            *reinterpret_cast<unsigned*>(mask_out + o) = mk;
        }
    } else {
        for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < n; i += stride) {
            int r = f.raw[i];
            bool bad = (r >= f.sat_adu) || (!f.pre && f.bpm && f.bpm[i] != 0);
            float c = f.pre ? calib_pre<false>((float)r, pre_load(f.offset, i, f.pre), pre_load(f.gain, i, f.pre), bad)
                            : calib_px((float)r, f.bias[i], f.dark[i], f.flat[i], bad, f.t_exp, f.flat_min);
            cal_out[i] = (c == c) ? c : 0.f;
            mask_out[i] = (c == c) ? 1 : 0;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// A6 standalone: sum[slot(idx[i])] += w v, wsum += w for a list of unique pixels.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) coadd_list_kernel(CoaddArgs ca, int ppt_log2, const long long* __restrict__ idx,
                                                        const float* __restrict__ value,
                                                        const float* __restrict__ weight, long long n) {
    long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    long long p = idx[i];
    long long key = p >> ppt_log2, lo = 0, hi = ca.n_tiles - 1, pos = -1;
    while (lo <= hi) {
        long long mid = (lo + hi) >> 1, tv = ca.tiles[mid];
        if (tv == key) { pos = mid; break; }
        if (tv < key) lo = mid + 1; else hi = mid - 1;
    }
    if (pos < 0) {
        if (ca.n_skipped) atomicAdd(ca.n_skipped, 1ull);
        return;
    }
    long long s = (pos << ppt_log2) + (p & ((1ll << ppt_log2) - 1));
    float wv = weight[i];
    ca.sum[s] = fmaf(wv, value[i], ca.sum[s]);
    ca.wsum[s] += wv;
}

// ------------------------------------------------------------------------------------------------
// pre-fused masters, once per pointing and exposure time (masters are uploaded at the
// start of each pointing).  offset = bias + dark * t_exp; gain = 1 / flat, NaN where the pixel is invalid (flat <
// flat_min or not finite, bias / dark not finite, bpm != 0, or not representable in the storage format).
// FMT: 1 float32, 2 binary16 (round to nearest even).  28 B in (+1 with a bpm), 8 or 4 B out per pixel.
// ------------------------------------------------------------------------------------------------
template <int FMT>
__global__ void __launch_bounds__(256) prepare_masters_kernel(const float* __restrict__ bias, const float* __restrict__ dark,
                                                             const float* __restrict__ flat, const unsigned char* __restrict__ bpm,
                                                             long long n, float t_exp, float flat_min, void* __restrict__ offset_out,
                                                             void* __restrict__ gain_out) {
    const long long stride = (long long)gridDim.x * 256;
    for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < n; i += stride) {
        const float b = bias[i], d = dark[i], fl = flat[i];
        float off = fmaf(d, t_exp, b);
        bool ok = (fl >= flat_min) && (fl < INFINITY) && (fabsf(b) < INFINITY) && (fabsf(d) < INFINITY) && !(bpm && bpm[i] != 0);
        float g = ok ? 1.0f / fl : nanf_();
        if (FMT == 1) {
            if (!(fabsf(off) < INFINITY)) { off = 0.f; g = nanf_(); }
            reinterpret_cast<float*>(offset_out)[i] = off;
            reinterpret_cast<float*>(gain_out)[i] = g;
        } else {
            __half ho = __float2half_rn(off), hg = __float2half_rn(g);
            if (!(fabsf(__half2float(ho)) < INFINITY) || (ok && !(fabsf(__half2float(hg)) < INFINITY))) {
                if (!(fabsf(__half2float(ho)) < INFINITY)) ho = __float2half_rn(0.f);
                hg = __float2half_rn(nanf_());
            }
            reinterpret_cast<__half*>(offset_out)[i] = ho;
            reinterpret_cast<__half*>(gain_out)[i] = hg;
        }
    }
}
