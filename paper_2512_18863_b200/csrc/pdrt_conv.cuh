// pdrt_conv.cuh — S3+S4+S5 fused (forward) and S8 (adjoint): the lateral pencil-kernel convolution.
//
// Forward (PAPER.md:123-133 Eq. 5-6, :145-149, :151-158 Eq. 8), per control point b and slice k:
//   Phivol(i,j) = mag^2 * bilinear_0(Phimap_b; mag u_i/Du + cuf, mag v_j/Dv + cvf),  mag = SID/(SID+w_k)
//   W_k         = lerp of the pre-integrated table W_tab at t = z_rad(b,k)/dz
//   D_b(i,j,k)  = sum_{dj,di} W_k[dj][di] * Phivol(i+di-c, j+dj-c)
// The projected fluence is never materialised: it is sampled straight into the shared-memory input
// tile.  Adjoint: H_b = conv of G_b with the flipped kernel, outputs restricted to S_k.
//
// This stage is bound by the FP32 FMA pipe (k^2 multiply-adds per 4-byte output), so the
// kernel is organised around FFMA issue slots: each thread owns an RU x RV = 8 x 4 register tile, slides
// a (K+7)-wide register window along u (LDS.128), and takes weights as warp-broadcast LDS.128; per input
// row that is (K+10)/4 + K loads for 32*K FFMAs.  Work items (control point, slice, chunk) come from
// device-built descriptors, so nothing about the aperture is known to or synchronised with the host;
// the grid is persistent (a multiple of the SM count) and strides over the item list.
#pragma once
#include "pdrt_dev.cuh"

namespace pdrt {

// Shared-memory tile columns are stored with an XOR swizzle on 16-byte quads: quad Q of a row lives at
// Q ^ ((Q >> 3) & 1).  Lanes tx and tx+4 of one row (32 floats apart, same banks) then hit different banks,
// so the LDS.128 window loads of 8 neighbouring thread-tiles are conflict-free.
__device__ __forceinline__ int swz_col(int c) { return c ^ (((c >> 5) & 1) << 2); }

__device__ __forceinline__ int find_cp(const int *__restrict__ tile_base, int n, int item)
{
    int lo = 0, hi = n;            // largest c with tile_base[c] <= item
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (tile_base[mid] <= item) lo = mid; else hi = mid;
    }
    return lo;
}

template <int KT, bool ADJ>
__global__ void __launch_bounds__(CONV_THREADS)
k_conv(Params P, const CpDesc *__restrict__ desc, int cp0, int n_cp, const int *__restrict__ tile_base,
       const float *__restrict__ phimap, const float *__restrict__ zrad, const float *__restrict__ wtab,
       const float *__restrict__ Gin, float *__restrict__ out)
{
    constexpr int C = (KT - 1) / 2;
    constexpr int KP = (KT + 3) & ~3;                 // weight row pitch [floats]
    constexpr int XW = (KT + RU - 1 + 3) & ~3;        // register window along u [floats]
    constexpr int NXQ = XW / 4;
    extern __shared__ float4 smem4[];
    float *Ws = reinterpret_cast<float *>(smem4);     // [KT][KP]
    float *tile = Ws + KT * KP;                       // [rows][pitch]
    const int tid = threadIdx.x;
    const int total = tile_base[n_cp];

    for (int item = blockIdx.x; item < total; item += gridDim.x) {
        const int slot = find_cp(tile_base, n_cp, item);
        const int cp = cp0 + slot;
        const CpDesc d = desc[cp];
        const int local = item - tile_base[slot];
        const int nch = d.ncx * d.ncy;
        const int k = local / nch, ch = local - k * nch;
        const int cy = ch / d.ncx, cx = ch - cy * d.ncx;
        // thread-tile range of this chunk inside the region
        const int ctx0 = cx * d.ntxc, ctx1 = min(d.ntx, ctx0 + d.ntxc);
        const int cty0 = cy * d.ntyc, cty1 = min(d.nty, cty0 + d.ntyc);
        const SliceBox S = slice_support(P, d, k);
        const SliceBox F = dilate(P, S, C);
        const SliceBox A = ADJ ? S : F;               // outputs to compute
        int atx0 = 0, atx1 = -1, aty0 = 0, aty1 = -1;
        if (!box_empty(A)) {
            atx0 = max(ctx0, (A.u0 - d.ri0) / RU); atx1 = min(ctx1 - 1, (A.u1 - d.ri0) / RU);
            aty0 = max(cty0, (A.v0 - d.rj0) / RV); aty1 = min(cty1 - 1, (A.v1 - d.rj0) / RV);
        }
        const bool active = atx0 <= atx1 && aty0 <= aty1;
        if (!ADJ) {
            // the resampler reads the whole compact region: thread-tiles outside F_k hold exact zeros
            const int cw = ctx1 - ctx0, chn = cw * (cty1 - cty0);
            for (int t = tid; t < chn; t += CONV_THREADS) {
                const int ty = cty0 + t / cw, tx = ctx0 + t % cw;
                if (active && tx >= atx0 && tx <= atx1 && ty >= aty0 && ty <= aty1) continue;
                const int i = d.ri0 + tx * RU;
#pragma unroll
                for (int jj = 0; jj < RV; ++jj) {
                    const int j = d.rj0 + ty * RV + jj;
                    if (j >= d.rj0 + d.pv) break;
                    float4 *o = reinterpret_cast<float4 *>(out + compact_index(P, d, slot, i, j, k));
                    o[0] = make_float4(0.f, 0.f, 0.f, 0.f);
                    o[1] = make_float4(0.f, 0.f, 0.f, 0.f);
                }
            }
        }
        if (!active) continue;                        // uniform across the block
        const int nax = atx1 - atx0 + 1, nay = aty1 - aty0 + 1;
        const int pitch = conv_pitch(KT, nax);
        const int rows = nay * RV + KT - 1;
        const int tu0 = d.ri0 + atx0 * RU - C, tv0 = d.rj0 + aty0 * RV - C;   // input coords of tile[0][0]

        // S4: slice kernel = lerp of the table in radiological depth (flipped for the adjoint)
        {
            const float t = zrad[(size_t)cp * P.Nw + k] / P.dz;
            int n0 = (int)floorf(t);
            n0 = min(max(n0, 0), P.n_z - 2);
            const float f = fminf(fmaxf(t - n0, 0.f), 1.f);
            const float *w0 = wtab + (size_t)n0 * KT * KT, *w1 = w0 + KT * KT;
            for (int e = tid; e < KT * KP; e += CONV_THREADS) {
                const int dj = e / KP, di = e - dj * KP;
                float v = 0.f;
                if (di < KT) {
                    const int src = ADJ ? (KT - 1 - dj) * KT + (KT - 1 - di) : dj * KT + di;
                    v = (1.f - f) * __ldg(w0 + src) + f * __ldg(w1 + src);
                }
                Ws[e] = v;
            }
        }
        // input tile: one warp per row, lanes along u (no integer division; coalesced for the adjoint)
        const int warp = tid >> 5, lane = tid & 31;
        if (!ADJ) {
            // S3: divergent projection of the fluence map, sampled on the fly (Eq. 5-6)
            const float mag = P.sid / (P.sid + P.wmin + k * P.dw), m2 = mag * mag;
            const float su = mag * P.du / P.Du, sv = mag / P.Dv;
            const float *pm = phimap + (size_t)cp * P.Nuf * P.Nvf;
            for (int r = warp; r < rows; r += CONV_THREADS / 32) {
                const int j = tv0 + r;
                float *trow = tile + r * pitch;
                if (j < S.v0 || j > S.v1) {
                    for (int c = lane; c < pitch; c += 32) trow[c] = 0.f;
                    continue;
                }
                const float fb = (P.v0 + j * P.dv) * sv + P.cvf;
                const float flb = floorf(fb);
                const int b = (int)flb;
                const float tb = fb - flb;
                const bool b0 = b >= d.b0 && b <= d.b1, b1 = b + 1 >= d.b0 && b + 1 <= d.b1;
                const float *pr0 = pm + b * P.Nuf, *pr1 = pr0 + P.Nuf;
                for (int c = lane; c < pitch; c += 32) {
                    const int i = tu0 + c;
                    float v = 0.f;
                    if (i >= S.u0 && i <= S.u1) {
                        const float fa = (i - P.cu) * su + P.cuf;
                        const float fla = floorf(fa);
                        const int a = (int)fla;
                        const float ta = fa - fla;
                        const bool a0 = a >= d.a0 && a <= d.a1, a1 = a + 1 >= d.a0 && a + 1 <= d.a1;
                        float s0 = 0.f, s1 = 0.f;
                        if (b0) s0 = (a0 ? (1.f - ta) * __ldg(pr0 + a) : 0.f) + (a1 ? ta * __ldg(pr0 + a + 1) : 0.f);
                        if (b1) s1 = (a0 ? (1.f - ta) * __ldg(pr1 + a) : 0.f) + (a1 ? ta * __ldg(pr1 + a + 1) : 0.f);
                        v = m2 * ((1.f - tb) * s0 + tb * s1);
                    }
                    trow[swz_col(c)] = v;
                }
            }
        } else {
            const int iend = min(d.ri0 + d.pu, P.Nu);
            for (int r = warp; r < rows; r += CONV_THREADS / 32) {
                const int j = tv0 + r;
                float *trow = tile + r * pitch;
                const bool rowin = j >= d.rj0 && j < d.rj0 + d.pv;
                const float *grow = Gin + (size_t)slot * (size_t)P.stride_cp + ((long long)(j - d.rj0) * P.Nw + k) * d.pu - d.ri0;
                for (int c = lane; c < pitch; c += 32) {
                    const int i = tu0 + c;
                    trow[swz_col(c)] = (rowin && i >= d.ri0 && i < iend) ? __ldg(grow + i) : 0.f;
                }
            }
        }
        __syncthreads();

        for (int t = tid; t < nax * nay; t += CONV_THREADS) {
            const int ty = t / nax, tx = t - ty * nax;
            float acc[RV][RU];
#pragma unroll
            for (int jj = 0; jj < RV; ++jj)
#pragma unroll
                for (int r = 0; r < RU; ++r) acc[jj][r] = 0.f;
            const float *xrow = tile + (ty * RV) * pitch;
            int xoff[NXQ];
#pragma unroll
            for (int q = 0; q < NXQ; ++q) xoff[q] = swz_col(tx * RU + 4 * q);
#pragma unroll 1
            for (int y = 0; y < KT + RV - 1; ++y) {
                float x[XW];
#pragma unroll
                for (int q = 0; q < NXQ; ++q) {
                    const float4 v = *reinterpret_cast<const float4 *>(xrow + xoff[q]);
                    x[4 * q] = v.x; x[4 * q + 1] = v.y; x[4 * q + 2] = v.z; x[4 * q + 3] = v.w;
                }
#pragma unroll
                for (int jj = 0; jj < RV; ++jj) {
                    const int dj = y - jj;
                    if (dj >= 0 && dj < KT) {
                        const float4 *w4 = reinterpret_cast<const float4 *>(Ws + dj * KP);
#pragma unroll
                        for (int q = 0; q < KP / 4; ++q) {
                            const float4 wv = w4[q];
                            const float w[4] = { wv.x, wv.y, wv.z, wv.w };
#pragma unroll
                            for (int e = 0; e < 4; ++e) {
                                const int di = 4 * q + e;
                                if (di < KT) {
#pragma unroll
                                    for (int r = 0; r < RU; ++r) acc[jj][r] = fmaf(w[e], x[r + di], acc[jj][r]);
                                }
                            }
                        }
                    }
                }
                xrow += pitch;
            }
            const int i = d.ri0 + (atx0 + tx) * RU;
#pragma unroll
            for (int jj = 0; jj < RV; ++jj) {
                const int j = d.rj0 + (aty0 + ty) * RV + jj;
                if (j < d.rj0 + d.pv) {
                    float4 *o = reinterpret_cast<float4 *>(out + compact_index(P, d, slot, i, j, k));
                    o[0] = make_float4(acc[jj][0], acc[jj][1], acc[jj][2], acc[jj][3]);
                    o[1] = make_float4(acc[jj][4], acc[jj][5], acc[jj][6], acc[jj][7]);
                }
            }
        }
        __syncthreads();
    }
}

// Expands the compact block of one control point to a dense [Nw][Nv][Nu] volume (stage tap for tests).
__global__ void k_expand_dense(Params P, const CpDesc *__restrict__ desc, int cp, int slot,
                               const float *__restrict__ comp, float *__restrict__ dense)
{
    const CpDesc d = desc[cp];
    const size_t n = (size_t)P.Nu * P.Nv * P.Nw;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(e % P.Nu), j = (int)((e / P.Nu) % P.Nv), k = (int)(e / ((size_t)P.Nu * P.Nv));
        float v = 0.f;
        if (d.a0 <= d.a1 && i >= d.ri0 && i < d.ri0 + d.pu && j >= d.rj0 && j < d.rj0 + d.pv)
            v = comp[compact_index(P, d, slot, i, j, k)];
        dense[e] = v;
    }
}

}  // namespace pdrt
