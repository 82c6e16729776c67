// common.cuh -- shared host/device declarations of the CUDA path (sm_100a).
//
// Geometry here is written in VECTOR form (unit vector of the HEALPix pixel centre, dot products with
// the tangent-plane basis at CRVAL); it is the product's own formulation and shares nothing with the
// oracle (which uses the angle form).  Citations: HEALPix nested scheme ref [10] PAPER.md:221;
// sky->pixel mapping PAPER.md:141; reprojection to the HEALPix grid PAPER.md:145.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define ARGUS_TILE_LOG2 5                 // output tile = 32 x 32 HEALPix pixels of one face
#define ARGUS_TILE_SIDE 32
#define ARGUS_TILE_PIX 1024               // = 1024 consecutive nested indices
#define ARGUS_MAX_COARSE 192              // coarse candidate cells passed by value to the scan kernel

// tile classes
#define TC_EMPTY 0
#define TC_INSIDE 1   // all 1024 pixels in the footprint; tile-local polynomial coordinates
#define TC_BORDER 2   // cut by the frame border; polynomial coordinates + per-pixel membership mask
#define TC_EXACT 3    // per-pixel FP64 coordinates (belt/cap ring, poles, cone edge, failed fit)

// Frame-constant projection data, computed on the host in FP64, passed to kernels by value.
struct DevWcs {
    double er[3], ee[3], en[3];  // radial / east / north unit vectors at CRVAL
    double m[2][2];              // (U,V) = m (xi, eta), xi/eta in radians  (= CD^-1 * 180/pi)
    double crpix[2];
    double cos_rho;              // cos(rho_max)
    double rho;                  // rho_max (rad)
    double ap[36], bp[36];
    int sip_order;
    int W, H;
    int k;                       // log2(nside)
    double nside;                // (double) nside
    double tile_ang;             // conservative angular radius of a 32x32 tile (rad)
};

// One output tile (32x32 HEALPix pixels).  x(s,t) = X0 + (ax*s + bx*t) * 2^-12 + Px(s/32, t/32) with
// s = 2u-31, t = 2v-31 the doubled, centred local pixel offsets (odd integers in [-31,31]); Px is a
// total-degree-3 polynomial, monomial order 1, S, T, S^2, ST, T^2, S^3, S^2 T, S T^2, T^3.
struct __align__(16) TileRec {
    long long tile;      // nested tile id = pixel index >> 10
    long long reserved;
    int cls;
    int count;
    int mask_slot;       // row of the membership-mask array (TC_BORDER / TC_EXACT), else -1
    int zone;            // 0 north cap, 1 belt, 2 south cap, -1 mixed
    int bx0, bx1, by0, by1;  // inclusive range of floor(x), floor(y) over the tile's member pixels
    int X0, Y0;
    int ax, bx, ay, by;
    float cx[10];
    float cy[10];
    int pad[2];
};

// Compact per-tile record of the TMA-staged bilinear kernel (resample_fast.cuh): 40 words = 10 x 16 B.
// Source position of the output pixel with doubled centred offsets (s, t) (odd integers in [-31, 31]),
// in units of 2^-24 px relative to the integer base (X0, Y0):
//   xf = c0x + ax*s + bx*t + float_as_int( P_x(s/32, t/32) )      (P_x already scaled by 2^24 and offset by
//   the 1.5*2^23 rounding constant, which c0x compensates);  cell = X0 + (xf >> 24), frac = (xf & (2^24-1)) 2^-24.
// The linear part is exact integer arithmetic; only the remainder (|.| < 0.22 px) is FP32.
#define FAST_FRAC_BITS 24
#define FAST_MAGIC_F 12582912.0f          // 1.5 * 2^23
#define FAST_MAGIC_I 0x4B400000
#define FAST_CAP_PX 3584                  // bilinear: staged source pixels per tile (box width x box rows), 2 stages
#define FAST_CAP_PX_LZ 4608               // Lanczos-3 (6x6 taps: 5 more rows and columns), 1 stage
                                          // the calibrated box (rows x bank-conflict-free pitch) may use cap * 9/8 floats
struct __align__(16) FastRec {
    int cls;             // TC_INSIDE / TC_BORDER when the tile is handled by the fast kernel, else 0
    int mask_slot;       // TC_BORDER: row of the membership-mask array
    int gx0, gy0;        // origin (cell) of the staged source box
    int wclass;          // bits 0..3: staged box width 40 + 8 w px (w = 0..4); bits 4..5: box rows 48 + 8 h (h = 0..3)
    int bh;              // rows of the box holding taps
    int kofs;            // (Y0 - gy0) * pitch + (X0 - gx0): cell -> calibrated-box index offset
    int X0;
    int c0x, ax, bx, c0y, ay, by;
    int Y0, poly_ok;     // poly_ok: the FP32 remainder stays inside the rounding-constant range
    float px[10];        // [0] = rounding constant, [1..9] monomials S, T, S^2, ST, T^2, S^3, S^2 T, S T^2, T^3
    float py[10];
    int pad2[4];
};
static_assert(sizeof(FastRec) == 160, "FastRec must be 10 x 16 bytes");

struct PlanStats {
    long long n_footprint, n_tiles, n_inside, n_border, n_exact, n_empty;
    int overflow;        // bit0: tile capacity, bit1: mask capacity, bit2: output capacity
    int pad;
};

struct CoarseList {
    int n;
    int ratio_log2;      // tile-level cells per coarse cell = 4^ratio_log2
    long long cell[ARGUS_MAX_COARSE];  // nested ids at the coarse resolution, ascending
};

// ------------------------------------------------------------------------------------------------
// HEALPix nested geometry (FP64, exact path)
// ------------------------------------------------------------------------------------------------
__host__ __device__ inline unsigned compact_even_bits(unsigned long long q) {
    q &= 0x5555555555555555ull;
    q = (q | (q >> 1)) & 0x3333333333333333ull;
    q = (q | (q >> 2)) & 0x0f0f0f0f0f0f0f0full;
    q = (q | (q >> 4)) & 0x00ff00ff00ff00ffull;
    q = (q | (q >> 8)) & 0x0000ffff0000ffffull;
    q = (q | (q >> 16)) & 0x00000000ffffffffull;
    return (unsigned)q;
}

__host__ __device__ inline void nest_to_xyf(long long p, int k, int& face, int& ix, int& iy) {
    unsigned long long q = (unsigned long long)p & ((1ull << (2 * k)) - 1ull);
    face = (int)(p >> (2 * k));
    ix = (int)compact_even_bits(q);
    iy = (int)compact_even_bits(q >> 1);
}

__host__ __device__ inline int face_ring_offset(int face) { return 2 + (face >> 2); }           // R_f
__host__ __device__ inline int face_phi_offset(int face) {                                       // P_f
    return (face >> 2) == 1 ? 2 * (face & 3) : 2 * (face & 3) + 1;
}

// zone of the integer ring number jr: 0 north cap (jr < nside), 1 belt, 2 south cap (jr > 3 nside)
__host__ __device__ inline int ring_zone(long long jr, long long nside) {
    return jr < nside ? 0 : (jr > 3 * nside ? 2 : 1);
}

#ifdef __CUDACC__
// Unit vector of the point (ix, iy) (real-valued, pixel centres at integers) of a face, using the
// formula of the given zone (so that a tile's formula can be continued half a pixel past its hull).
__device__ inline void hp_vec(int face, double ix, double iy, double nside, int zone, double v[3]) {
    double jr = (double)face_ring_offset(face) * nside - ix - iy - 1.0;
    double z, sth, nr;
    if (zone == 1) {
        nr = nside;
        z = (2.0 / 3.0) * (2.0 - jr / nside);
        sth = sqrt((1.0 - z) * (1.0 + z));
    } else {
        nr = (zone == 0) ? jr : 4.0 * nside - jr;
        double t = nr * nr / (3.0 * nside * nside);
        z = (zone == 0) ? 1.0 - t : t - 1.0;
        sth = sqrt(t * (2.0 - t));
    }
    double s, c;
    sincospi(0.25 * ((double)face_phi_offset(face) + (ix - iy) / nr), &s, &c);
    v[0] = sth * c;
    v[1] = sth * s;
    v[2] = z;
}

// Sky direction -> frame pixel coordinates (inverse TAN + sky->pixel SIP).  Returns cos c.
__device__ inline double vec_to_xy(const DevWcs& w, const double v[3], double& x, double& y) {
    double cosc = v[0] * w.er[0] + v[1] * w.er[1] + v[2] * w.er[2];
    double inv = 1.0 / cosc;
    double xi = (v[0] * w.ee[0] + v[1] * w.ee[1] + v[2] * w.ee[2]) * inv;
    double eta = (v[0] * w.en[0] + v[1] * w.en[1] + v[2] * w.en[2]) * inv;
    double U = w.m[0][0] * xi + w.m[0][1] * eta;
    double V = w.m[1][0] * xi + w.m[1][1] * eta;
    double fu = 0.0, fv = 0.0;
    if (w.sip_order > 0) {
        double up = 1.0;
        for (int p = 0; p <= w.sip_order; ++p) {
            double m = up;
            for (int q = 0; p + q <= w.sip_order; ++q) {
                fu = fma(w.ap[p * 6 + q], m, fu);
                fv = fma(w.bp[p * 6 + q], m, fv);
                m *= V;
            }
            up *= U;
        }
    }
    x = U + fu + w.crpix[0];
    y = V + fv + w.crpix[1];
    return cosc;
}

// Exact per-pixel mapping of an integer pixel (face, ix, iy).  Returns cos c.
__device__ inline double pixel_to_xy(const DevWcs& w, int face, int ix, int iy, double& x, double& y) {
    long long ns = 1ll << w.k;
    long long jr = (long long)face_ring_offset(face) * ns - ix - iy - 1;
    double v[3];
    hp_vec(face, (double)ix, (double)iy, w.nside, ring_zone(jr, ns), v);
    return vec_to_xy(w, v, x, y);
}

// Footprint predicate on exact coordinates (half-open domain, PAPER-silent reading in DESIGN.md).
__device__ inline bool in_domain(const DevWcs& w, double cosc, double x, double y) {
    return (cosc >= w.cos_rho) && (x >= -0.5) && (x < (double)w.W - 0.5) && (y >= -0.5) && (y < (double)w.H - 0.5);
}

// ------------------------------------------------------------------------------------------------
// Tile-local FP32 coordinates: integer cell (i0, j0) and fractions (fx, fy) of the source position.
// The dominant linear part is carried exactly in 20.12 fixed point, the remainder (|.| < ~1.1) in FP32:
// absolute error ~1.5e-7 px.
// ------------------------------------------------------------------------------------------------
struct PolyAxis {
    float c0, c1, c2, c3, c4, c5, c6, c7, c8, c9;
    int base, a, b;
};

__device__ inline void poly_axis_load(const TileRec& r, int axis, PolyAxis& p) {
    const float* c = axis ? r.cy : r.cx;
    p.c0 = c[0]; p.c1 = c[1]; p.c2 = c[2]; p.c3 = c[3]; p.c4 = c[4];
    p.c5 = c[5]; p.c6 = c[6]; p.c7 = c[7]; p.c8 = c[8]; p.c9 = c[9];
    p.base = axis ? r.Y0 : r.X0;
    p.a = axis ? r.ay : r.ax;
    p.b = axis ? r.by : r.bx;
}

// s, t: odd integers in [-31, 31]
__device__ inline void poly_axis_eval(const PolyAxis& p, int s, int t, int& cell, float& frac) {
    float S = (float)s * 0.03125f, T = (float)t * 0.03125f;
    float A = fmaf(S, fmaf(S, fmaf(S, p.c6, p.c3), p.c1), p.c0);
    float B = fmaf(S, fmaf(S, p.c7, p.c4), p.c2);
    float C = fmaf(S, p.c8, p.c5);
    float lo = fmaf(T, fmaf(T, fmaf(T, p.c9, C), B), A);
    int hi = p.a * s + p.b * t;                       // exact, units of 2^-12 px
    float g = fmaf((float)(hi & 4095), 0.000244140625f, lo);
    float fl = floorf(g);
    frac = g - fl;
    cell = p.base + (hi >> 12) + (int)fl;
}

// Same coordinates with the remainder polynomial evaluated in FP64 from the unsplit double coefficients
// dc[10] (constant term includes the integer base): used by the Lanczos-3 path (error ~1e-10 px).
__device__ inline void poly_axis_eval_f64(const double* __restrict__ dc, const PolyAxis& p, int s, int t, int& cell,
                                          double& frac) {
    double S = (double)s * 0.03125, T = (double)t * 0.03125;
    // remove the fixed-point linear part and the integer base exactly, as in the FP32 split
    double c0 = dc[0] - (double)p.base, c1 = dc[1] - (double)p.a * (32.0 / 4096.0), c2 = dc[2] - (double)p.b * (32.0 / 4096.0);
    double A = fma(S, fma(S, fma(S, dc[6], dc[3]), c1), c0);
    double B = fma(S, fma(S, dc[7], dc[4]), c2);
    double C = fma(S, dc[8], dc[5]);
    double lo = fma(T, fma(T, fma(T, dc[9], C), B), A);
    int hi = p.a * s + p.b * t;
    double g = fma((double)(hi & 4095), 0.000244140625, lo);
    double fl = floor(g);
    frac = g - fl;
    cell = p.base + (hi >> 12) + (int)fl;
}
#endif  // __CUDACC__

// ---- packed FP32 (Blackwell FFMA2 / FMUL2 / FADD2: two IEEE operations per instruction, either operand may be a scalar
// broadcast).  The clean interpolation loops are bound by instruction issue, and their x and y halves (and neighbouring rows
// of taps) run the same operations on different data: packed, the Lanczos-3 weights + gather take 60 instructions less per
// output.  Each lane of a packed operation rounds exactly as the scalar one: results are bit-identical to the scalar form.
#ifndef ARGUS_NO_F32X2
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) {
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(*reinterpret_cast<unsigned long long*>(&a)), "l"(*reinterpret_cast<unsigned long long*>(&b)),
        "l"(*reinterpret_cast<unsigned long long*>(&c)));
    return *reinterpret_cast<float2*>(&d);
}
__device__ __forceinline__ float2 mul2(float2 a, float2 b) {
    unsigned long long d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(*reinterpret_cast<unsigned long long*>(&a)), "l"(*reinterpret_cast<unsigned long long*>(&b)));
    return *reinterpret_cast<float2*>(&d);
}
__device__ __forceinline__ float2 add2(float2 a, float2 b) {
    unsigned long long d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(*reinterpret_cast<unsigned long long*>(&a)), "l"(*reinterpret_cast<unsigned long long*>(&b)));
    return *reinterpret_cast<float2*>(&d);
}
#else
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return make_float2(fmaf(a.x, b.x, c.x), fmaf(a.y, b.y, c.y)); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return make_float2(__fmul_rn(a.x, b.x), __fmul_rn(a.y, b.y)); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return make_float2(__fadd_rn(a.x, b.x), __fadd_rn(a.y, b.y)); }
#endif
__device__ __forceinline__ float2 bc2(float s) { return make_float2(s, s); }

