// subtract.cuh -- direct image subtraction per tile on the tile-dense HEALPix grid (DESIGN.md
// section 13): the step the paper runs on the CPU at 20 ms per tile and names "a GPU implementation is in development"
// (PAPER.md:163 sec. 5.2, :185, :201 Table 2).  The paper gives no formula (ref [17]); readings R-X1 .. R-X8 of
// DESIGN.md are restated in include/argus.h.  Both images are (sum, wsum) pairs in the argus_coadd layout, as
// argus_resample_coadd writes them: image = sum / wsum.
//
//   sub_stats_kernel   per tile slice: n, sum r, sum s, sum r r, sum r s over the valid pixels, FP64, one partial per CTA
//                      (fixed summation order: the fit is deterministic)
//   sub_fit_kernel     per tile: partials -> (alpha, beta) of the least-squares match s ~ alpha r + beta (R-X2)
//   sub_tiles_kernel   per 32 x 32-pixel block (1024 consecutive nested indices): difference, noise, significance
//                      (R-X3 .. R-X5) with 128-bit loads and stores; significance + difference of the block and its
//                      one-pixel apron in shared memory; thresholded local maxima with the nested-index tie rule (R-X6),
//                      records in nested order at an atomically reserved base (R-X7)
//   det_scan_kernel    (background.cuh) exclusive scan of the per-block counts
//   sub_gather_kernel  one warp per block copies its records to their final position (R-X8: ascending nested index)
#pragma once
#include "background.cuh"

#define SUB_SPLIT_MAX 32             // CTAs per tile in the statistics pass
#define SUB_BLOCK 1024               // pixels per detection block = 32 x 32 = 1024 consecutive nested indices
#define SUB_PITCH 35                 // shared grid pitch (34 + 1: odd, so that the 2 x 2 stores spread over the banks)

struct ArgusTransientRec {           // == argus_transient (argus.h)
    long long pixel;
    float sig, diff, flux, noise;
    int tile_rank, reserved;
};

struct SubParams {
    int match, n_min;
    float sci_wmin, ref_wmin, rn2, inv_gain, k_sigma;
};

__device__ __forceinline__ unsigned spread_bits16(unsigned v) {       // bit i -> bit 2 i (16 bits)
    v &= 0xffffu;
    v = (v | (v << 8)) & 0x00ff00ffu;
    v = (v | (v << 4)) & 0x0f0f0f0fu;
    v = (v | (v << 2)) & 0x33333333u;
    v = (v | (v << 1)) & 0x55555555u;
    return v;
}

// The two images at one pixel: s = sum / wsum through one reciprocal each (rcp.approx: 1 ulp, so the quotients are within 2 ulp =
// 2.4e-7 relative, 40 x inside the 1e-5 relative tolerance; the weights are >= wmin > 0).  Both passes use these same float32
// values: the fit is made on the images the difference is formed from.
__device__ __forceinline__ void sub_images(float ssv, float swv, float rsv, float rwv, float& s, float& r, float& isw, float& irw) {
    isw = rcp_ftz(swv); irw = rcp_ftz(rwv);
    s = ssv * isw; r = rsv * irw;
}
__device__ __forceinline__ float rsqrt_ftz(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// ---------------------------------------------------------------------------------------------- statistics
// grid = (tiles of the chunk) * split CTAs of 256 threads; CTA (t, j) covers pixels [j, j + 1) * ppt / split of tile tile0 + t.
__global__ void __launch_bounds__(256) sub_stats_kernel(const float* __restrict__ ss, const float* __restrict__ sw,
                                                       const float* __restrict__ rs, const float* __restrict__ rw,
                                                       long long ppt, int split, long long tile0, SubParams p, double* __restrict__ partial) {
    __shared__ double s_red[8][5];
    const long long tile = tile0 + blockIdx.x / split;
    const int j = blockIdx.x % split;
    const long long n4 = (ppt / split) >> 2;                    // float4 items of this slice (ppt / split >= 1024 / 32 ...)
    const size_t base = (size_t)tile * ppt + (size_t)j * (ppt / split);
    const float4* a = reinterpret_cast<const float4*>(ss + base);
    const float4* b = reinterpret_cast<const float4*>(sw + base);
    const float4* c = reinterpret_cast<const float4*>(rs + base);
    const float4* d = reinterpret_cast<const float4*>(rw + base);
    double acc[5] = {0, 0, 0, 0, 0};
    for (long long i = threadIdx.x; i < n4; i += 256) {
        const float4 x = __ldg(a + i), wx = __ldg(b + i), y = __ldg(c + i), wy = __ldg(d + i);
        const float xs[4] = {x.x, x.y, x.z, x.w}, ws[4] = {wx.x, wx.y, wx.z, wx.w};
        const float ys[4] = {y.x, y.y, y.z, y.w}, wr[4] = {wy.x, wy.y, wy.z, wy.w};
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (ws[k] >= p.sci_wmin && wr[k] >= p.ref_wmin) {
                float sf, rf, i0, i1;
                sub_images(xs[k], ws[k], ys[k], wr[k], sf, rf, i0, i1);                  // the float32 images the subtraction uses
                const double s = (double)sf, r = (double)rf;
                acc[0] += 1.0; acc[1] += r; acc[2] += s; acc[3] += r * r; acc[4] += r * s;
            }
        }
    }
#pragma unroll
    for (int k = 0; k < 5; ++k)
        for (int o = 16; o; o >>= 1) acc[k] += __shfl_xor_sync(0xffffffffu, acc[k], o);
    if ((threadIdx.x & 31) == 0)
        for (int k = 0; k < 5; ++k) s_red[threadIdx.x >> 5][k] = acc[k];
    __syncthreads();
    if (threadIdx.x < 5) {
        double t = 0;
        for (int w = 0; w < 8; ++w) t += s_red[w][threadIdx.x];
        partial[((size_t)tile * SUB_SPLIT_MAX + j) * 5 + threadIdx.x] = t;
    }
}

// R-X2.  One thread per tile.  fit[t] = (alpha, beta) as floats for the per-pixel pass.
__global__ void sub_fit_kernel(const double* __restrict__ partial, long long tile0, long long n_tiles, int split, SubParams p, int have_stats,
                               float2* __restrict__ fit, float* __restrict__ alpha_out, float* __restrict__ beta_out,
                               int* __restrict__ nvalid_out) {
    const long long t = tile0 + (long long)blockIdx.x * blockDim.x + threadIdx.x;     // tiles [tile0, n_tiles) of this chunk
    if (t >= n_tiles) return;
    double alpha = 1.0, beta = 0.0, n = 0;
    if (have_stats) {
        double S[5] = {0, 0, 0, 0, 0};
        for (int j = 0; j < split; ++j)
            for (int k = 0; k < 5; ++k) S[k] += partial[((size_t)t * SUB_SPLIT_MAX + j) * 5 + k];
        n = S[0];
        if (p.match == 1 && n > 0) {
            const double den = n * S[3] - S[1] * S[1];
            if (n >= (double)p.n_min && den > 1e-10 * n * S[3]) {   // a reference without structure has no slope (R-X2)
                alpha = (n * S[4] - S[1] * S[2]) / den;
                beta = (S[2] - alpha * S[1]) / n;
            } else {
                beta = (S[2] - S[1]) / n;
            }
        }
    }
    fit[t] = make_float2((float)alpha, (float)beta);
    if (alpha_out) alpha_out[t] = (float)alpha;
    if (beta_out) beta_out[t] = (float)beta;
    if (nvalid_out) nvalid_out[t] = (int)n;
}

// ---------------------------------------------------------------------------------------------- per pixel
// R-X1, R-X3 .. R-X5 for one pixel.  Invalid: d = 0, S = -inf (never a maximum).  Five IEEE divisions and a square root per
// pixel made this pass instruction-bound (XU pipe 34 %, 128 instructions per pixel); two reciprocals and one reciprocal
// square root (2 ulp each; the variance is > 0: read noise > 0) leave every output within 1e-6 relative of the IEEE form.
__device__ __forceinline__ void sub_px(float ssv, float swv, float rsv, float rwv, const SubParams& p, float alpha, float beta,
                                       float& d, float& S, float& sigma) {
    d = 0.f; sigma = 0.f; S = __int_as_float(0xff800000);
    if (swv >= p.sci_wmin && rwv >= p.ref_wmin) {
        float s, r, isw, irw;
        sub_images(ssv, swv, rsv, rwv, s, r, isw, irw);
        const float m = fmaf(alpha, r, beta);
        d = s - m;
        const float var = (p.rn2 + fmaxf(m, 0.f) * p.inv_gain) * fmaf(alpha * alpha, irw, isw);
        const float rs = rsqrt_ftz(var);
        sigma = var * rs;
        S = d * rs;
    }
}

// grid-stride over blocks of 1024 consecutive nested indices; 256 threads, thread t <-> in-block indices 4 t .. 4 t + 3
// (a 2 x 2 pixel group: one 128-bit load per array, one 128-bit store per output).
#ifndef SUB_TILES_MINB
#define SUB_TILES_MINB 6                 // 39 registers, 16 B of spills: six CTAs per SM hide the load latency (4: 0.452, 5: 0.427, 6: 0.421, 8: 0.487 ms per call)
#endif
__global__ void __launch_bounds__(256, SUB_TILES_MINB) sub_tiles_kernel(const float* __restrict__ ss, const float* __restrict__ sw,
                                                       const float* __restrict__ rs, const float* __restrict__ rw,
                                                       const long long* __restrict__ tiles, long long ppt, int side_log2,
                                                       long long b0, long long n_blocks, SubParams p, const float2* __restrict__ fit,
                                                       float* __restrict__ diff_out, float* __restrict__ sig_out,
                                                       ArgusTransientRec* __restrict__ tmp, unsigned capacity,
                                                       uint2* __restrict__ block_info, unsigned* __restrict__ total) {
    __shared__ float s_S[34 * SUB_PITCH], s_d[34 * SUB_PITCH];
    __shared__ int s_warp[8];
    __shared__ unsigned s_base;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const int bpt_log2 = 2 * side_log2 - 10;                      // blocks per tile = ppt / 1024
    const int side = 1 << side_log2;
    const int gx = 2 * (int)compact_even_bits((unsigned)tid), gy = 2 * (int)compact_even_bits((unsigned)tid >> 1);   // 2 x 2 group origin
    const float ninf = __int_as_float(0xff800000);
    for (long long b = b0 + blockIdx.x; b < n_blocks; b += gridDim.x) {      // blocks [b0, n_blocks) of this chunk
        const long long tile = b >> bpt_log2;
        const unsigned bi = (unsigned)(b & ((1ll << bpt_log2) - 1));
        const int Bx = 32 * (int)compact_even_bits(bi), By = 32 * (int)compact_even_bits(bi >> 1);
        const float2 ab = __ldg(fit + tile);
        const size_t o = (size_t)b * SUB_BLOCK + 4 * tid;
        const float4 a4 = __ldg(reinterpret_cast<const float4*>(ss + o)), b4 = __ldg(reinterpret_cast<const float4*>(sw + o));
        const float4 c4 = __ldg(reinterpret_cast<const float4*>(rs + o)), d4 = __ldg(reinterpret_cast<const float4*>(rw + o));
        float d[4], S[4], sg[4];
        sub_px(a4.x, b4.x, c4.x, d4.x, p, ab.x, ab.y, d[0], S[0], sg[0]);
        sub_px(a4.y, b4.y, c4.y, d4.y, p, ab.x, ab.y, d[1], S[1], sg[1]);
        sub_px(a4.z, b4.z, c4.z, d4.z, p, ab.x, ab.y, d[2], S[2], sg[2]);
        sub_px(a4.w, b4.w, c4.w, d4.w, p, ab.x, ab.y, d[3], S[3], sg[3]);
        *reinterpret_cast<float4*>(diff_out + o) = make_float4(d[0], d[1], d[2], d[3]);
        if (sig_out)
            *reinterpret_cast<float4*>(sig_out + o) = make_float4(S[0] == ninf ? 0.f : S[0], S[1] == ninf ? 0.f : S[1],
                                                                  S[2] == ninf ? 0.f : S[2], S[3] == ninf ? 0.f : S[3]);
        __syncthreads();                                            // previous block's readers are done with the grids
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const int x = gx + (k & 1), y = gy + (k >> 1);
            s_S[(y + 1) * SUB_PITCH + x + 1] = S[k];
            s_d[(y + 1) * SUB_PITCH + x + 1] = d[k];
        }
        if (tid < 132) {                                            // one-pixel apron, from the neighbouring blocks of the SAME tile
            int x, y;
            if (tid < 34) { x = tid - 1; y = -1; }
            else if (tid < 68) { x = tid - 35; y = 32; }
            else if (tid < 100) { x = -1; y = tid - 68; }
            else { x = 32; y = tid - 100; }
            const int X = Bx + x, Y = By + y;
            float dd = 0.f, SS = ninf, sgm;
            if (X >= 0 && X < side && Y >= 0 && Y < side) {
                const size_t q = (size_t)tile * ppt + (spread_bits16((unsigned)X) | (spread_bits16((unsigned)Y) << 1));
                sub_px(__ldg(ss + q), __ldg(sw + q), __ldg(rs + q), __ldg(rw + q), p, ab.x, ab.y, dd, SS, sgm);
            }
            s_S[(y + 1) * SUB_PITCH + x + 1] = SS;
            s_d[(y + 1) * SUB_PITCH + x + 1] = dd;
        }
        __syncthreads();
        // R-X6: threshold first (rare), then the 8-neighbour test with the nested-index tie rule
        unsigned bits = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (S[k] > p.k_sigma) {
                const int x = gx + (k & 1), y = gy + (k >> 1);
                const unsigned qp = spread_bits16((unsigned)(Bx + x)) | (spread_bits16((unsigned)(By + y)) << 1);
                bool is_max = true;
#pragma unroll
                for (int dy = -1; dy <= 1; ++dy)
#pragma unroll
                    for (int dx = -1; dx <= 1; ++dx) {
                        if (dx == 0 && dy == 0) continue;
                        const float Sn = s_S[(y + 1 + dy) * SUB_PITCH + x + 1 + dx];
                        const unsigned qn = spread_bits16((unsigned)(Bx + x + dx)) | (spread_bits16((unsigned)(By + y + dy)) << 1);
                        is_max = is_max && (qn < qp ? S[k] > Sn : S[k] >= Sn);   // outside the tile: Sn = -inf
                    }
                if (is_max) bits |= 1u << k;
            }
        }
        const int cnt = __popc(bits);
        int inc = cnt;
#pragma unroll
        for (int o2 = 1; o2 < 32; o2 <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, inc, o2);
            if (lane >= o2) inc += v;
        }
        if (lane == 31) s_warp[wid] = inc;
        __syncthreads();
        int before = inc - cnt, block_cnt = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) {
            const int c = s_warp[w];
            before += (w < wid) ? c : 0;
            block_cnt += c;
        }
        if (tid == 0) {
            const unsigned base = block_cnt ? atomicAdd(total, (unsigned)block_cnt) : 0u;
            block_info[b] = make_uint2(base, (unsigned)block_cnt);
            s_base = base;
        }
        if (block_cnt == 0) continue;                               // uniform over the CTA
        __syncthreads();
        unsigned pos = s_base + (unsigned)before;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (!((bits >> k) & 1u)) continue;
            const int x = gx + (k & 1), y = gy + (k >> 1);
            float flux = 0.f;
#pragma unroll
            for (int dy = -1; dy <= 1; ++dy)
#pragma unroll
                for (int dx = -1; dx <= 1; ++dx) flux += s_d[(y + 1 + dy) * SUB_PITCH + x + 1 + dx];   // invalid / outside: 0
            if (pos < capacity) {
                ArgusTransientRec rec;
                rec.pixel = __ldg(tiles + tile) * ppt + (long long)(bi * SUB_BLOCK + 4 * tid + k);
                rec.sig = S[k]; rec.diff = d[k]; rec.flux = flux; rec.noise = sg[k];
                rec.tile_rank = (int)tile; rec.reserved = 0;
                uint4* dst = reinterpret_cast<uint4*>(tmp + pos);
                const uint4* src = reinterpret_cast<const uint4*>(&rec);
                dst[0] = src[0];
                dst[1] = src[1];
            }
            ++pos;
        }
    }
}

// One warp per block: tmp[base .. base + cnt) -> out[offset .. offset + cnt)  (blocks are in ascending nested order).
__global__ void __launch_bounds__(256) sub_gather_kernel(const uint2* __restrict__ block_info, const unsigned* __restrict__ offsets,
                                                        long long n_blocks, const ArgusTransientRec* __restrict__ tmp,
                                                        ArgusTransientRec* __restrict__ out, unsigned capacity) {
    const long long b = (long long)blockIdx.x * 8 + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (b >= n_blocks) return;
    const uint2 info = block_info[b];
    const unsigned off = offsets[b];
    for (unsigned j = lane; j < info.y; j += 32) {
        if (info.x + j >= capacity || off + j >= capacity) break;
        const uint4* src = reinterpret_cast<const uint4*>(tmp + info.x + j);
        uint4* dst = reinterpret_cast<uint4*>(out + off + j);
        dst[0] = src[0];
        dst[1] = src[1];
    }
}
