// pdrt_conv.cuh — S3+S4+S5 fused (forward) and S7+S8 fused (adjoint): the lateral pencil-kernel convolution.
//
// Forward (PAPER.md:123-133 Eq. 5-6, :145-149, :151-158 Eq. 8), per control point b and slice k:
//   Phivol(i,j) = mag^2 * bilinear_0(Phimap_b; mag u_i/Du + cuf, mag v_j/Dv + cvf),  mag = SID/(SID+w_k)
//   W_k         = lerp of the pre-integrated table W_tab at t = z_rad(b,k)/dz
//   D_b(i,j,k)  = sum_{dj,di} W_k[dj][di] * Phivol(i+di-c, j+dj-c)
// The projected fluence is never materialised: it is sampled straight into the shared-memory input tile.
//
// Adjoint (transposes of Eq. 9 and Eq. 8): G_b = R_b^T g is never materialised either.  The gantry rotates
// about patient z = beam v, so the bilinear weights of a beam voxel (i,k) onto the patient voxels (x,y) of
// its rotated unit hat do not depend on v: one warp fills one tile row (fixed i, lanes along v), computes
// the handful of weights once and streams coalesced reads of gT[y][x][v].  Then H_b = conv of G_b with the
// flipped kernel, outputs restricted to S_k.
//
// The convolution is bound by the FP32 FMA pipe (k^2 multiply-adds per 4-byte output), so the
// kernel is organised around FFMA issue slots: each thread owns an RF x RS = 8(v) x 2(u) register tile,
// slides a (K+7)-wide register window along v (LDS.128), and takes weights as warp-broadcast LDS.128.
// Work items (control point, slice, chunk) come from device-built descriptors, so nothing about the
// aperture is known to or synchronised with the host; the grid is persistent (a multiple of the SM count)
// and strides over the item list.
#pragma once
#include "pdrt_dev.cuh"

namespace pdrt {

// Shared-memory tile columns are stored with an XOR swizzle on 16-byte quads: quad Q of a row lives at
// Q ^ ((Q >> 3) & 1).  Lanes tf and tf+4 of one row (32 floats apart, same banks) then hit different banks,
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
       const float *__restrict__ phimapT, const float *__restrict__ zrad, const float *__restrict__ wtab,
       const float *__restrict__ gT, float *__restrict__ out)
{
    constexpr int C = (KT - 1) / 2;
    constexpr int KP = (KT + 3) & ~3;                 // weight row pitch [floats]
    constexpr int XW = (KT + RF - 1 + 3) & ~3;        // register window along v [floats]
    constexpr int NXQ = XW / 4;
    constexpr int PMAX = (NTFC_MAX * RF + XW - RF + 7) & ~7;   // widest tile row
    constexpr int MC = (PMAX + 31) / 32;              // tile columns per lane in the adjoint fill
    extern __shared__ float4 smem4[];
    float *Ws = reinterpret_cast<float *>(smem4);     // [KT (du)][KP (dv)]
    float *tile = Ws + KT * KP;                       // [rows along u][pitch along v]
    const int tid = threadIdx.x;
    const int total = tile_base[n_cp];

    for (int item = blockIdx.x; item < total; item += gridDim.x) {
        const int slot = find_cp(tile_base, n_cp, item);
        const int cp = cp0 + slot;
        const CpDesc d = desc[cp];
        const int local = item - tile_base[slot];
        const int nch = d.ncf * d.ncs;
        const int k = local / nch, ch = local - k * nch;
        const int cs = ch / d.ncf, cf = ch - cs * d.ncf;
        // thread-tile range of this chunk inside the region
        const int ctf0 = cf * d.ntfc, ctf1 = min(d.ntf, ctf0 + d.ntfc);
        const int cts0 = cs * d.ntsc, cts1 = min(d.nts, cts0 + d.ntsc);
        const SliceBox S = slice_support(P, d, k);
        const SliceBox F = dilate(P, S, C);
        const SliceBox A = ADJ ? S : F;               // outputs to compute
        int atf0 = 0, atf1 = -1, ats0 = 0, ats1 = -1;
        if (!box_empty(A)) {
            atf0 = max(ctf0, (A.v0 - d.rj0) / RF); atf1 = min(ctf1 - 1, (A.v1 - d.rj0) / RF);
            ats0 = max(cts0, (A.u0 - d.ri0) / RS); ats1 = min(cts1 - 1, (A.u1 - d.ri0) / RS);
        }
        const bool active = atf0 <= atf1 && ats0 <= ats1;
        float *oslice = out + (size_t)slot * (size_t)P.stride_cp + (size_t)k * d.pu * d.pv;   // [pu][pv] of slice k
        if (!ADJ) {
            // the resampler reads the whole compact region: thread-tiles outside F_k hold exact zeros
            const int cw = ctf1 - ctf0, chn = cw * (cts1 - cts0);
            for (int t = tid; t < chn; t += CONV_THREADS) {
                const int ts = cts0 + t / cw, tf = ctf0 + t % cw;
                if (active && tf >= atf0 && tf <= atf1 && ts >= ats0 && ts <= ats1) continue;
#pragma unroll
                for (int ii = 0; ii < RS; ++ii) {
                    float4 *o = reinterpret_cast<float4 *>(oslice + (size_t)(ts * RS + ii) * d.pv + tf * RF);
                    o[0] = make_float4(0.f, 0.f, 0.f, 0.f);
                    o[1] = make_float4(0.f, 0.f, 0.f, 0.f);
                }
            }
        }
        if (!active) continue;                        // uniform across the block
        const int naf = atf1 - atf0 + 1, nas = ats1 - ats0 + 1;
        const int pitch = conv_pitch(KT, naf);
        const int rows = nas * RS + KT - 1;
        const int tv0 = d.rj0 + atf0 * RF - C, tu0 = d.ri0 + ats0 * RS - C;   // input coords of tile[0][0]

        // S4: slice kernel = lerp of the table in radiological depth, stored [du][dv] (flipped for the adjoint)
        {
            const float t = zrad[(size_t)cp * P.Nw + k] / P.dz;
            int n0 = (int)floorf(t);
            n0 = min(max(n0, 0), P.n_z - 2);
            const float f = fminf(fmaxf(t - n0, 0.f), 1.f);
            const float *w0 = wtab + (size_t)n0 * KT * KT, *w1 = w0 + KT * KT;
            for (int e = tid; e < KT * KP; e += CONV_THREADS) {
                const int di = e / KP, dj = e - di * KP;
                float v = 0.f;
                if (dj < KT) {
                    const int src = ADJ ? (KT - 1 - dj) * KT + (KT - 1 - di) : dj * KT + di;
                    v = (1.f - f) * __ldg(w0 + src) + f * __ldg(w1 + src);
                }
                Ws[e] = v;
            }
        }
        // input tile: one warp per row (fixed u index), lanes along v
        const int warp = tid >> 5, lane = tid & 31;
        if (!ADJ) {
            // S3: divergent projection of the fluence map, sampled on the fly (Eq. 5-6)
            const float mag = P.sid / (P.sid + P.wmin + k * P.dw), m2 = mag * mag;
            const float su = mag * P.du / P.Du, sv = mag / P.Dv;
            const float *pm = phimapT + (size_t)cp * P.Nuf * P.Nvf;
            // per-column terms (v index, interpolation fraction, validity) do not depend on the row: once per item
            int cb[MC];
            float ctb[MC];
#pragma unroll
            for (int m = 0; m < MC; ++m) {
                const int j = tv0 + lane + 32 * m;
                const float fb = (P.v0 + j * P.dv) * sv + P.cvf;
                const float flb = floorf(fb);
                const int b = (int)flb;
                ctb[m] = fb - flb;
                const bool jin = lane + 32 * m < pitch && j >= S.v0 && j <= S.v1;
                const bool b0 = jin && b >= d.b0 && b <= d.b1, b1 = jin && b + 1 >= d.b0 && b + 1 <= d.b1;
                cb[m] = (b0 || b1) ? (((b + 1) << 2) | (b0 ? 1 : 0) | (b1 ? 2 : 0)) : 0;     // b >= -1 when a flag is set
            }
            for (int r = warp; r < rows; r += CONV_THREADS / 32) {
                const int i = tu0 + r;
                float *trow = tile + r * pitch;
                if (i < S.u0 || i > S.u1) {
                    for (int c = lane; c < pitch; c += 32) trow[c] = 0.f;
                    continue;
                }
                const float fa = (i - P.cu) * su + P.cuf;
                const float fla = floorf(fa);
                const int a = (int)fla;
                const float ta = fa - fla;
                const bool a0 = a >= d.a0 && a <= d.a1, a1 = a + 1 >= d.a0 && a + 1 <= d.a1;
                const float wa0 = a0 ? 1.f - ta : 0.f, wa1 = a1 ? ta : 0.f;
                // invalid rows of the map get weight 0 and are folded onto a valid one, so every address is readable
                const float *pc0 = pm + (a0 ? a : a + 1) * P.Nvf, *pc1 = pm + (a1 ? a + 1 : a) * P.Nvf;
                const bool arow = a0 || a1;
#pragma unroll
                for (int m = 0; m < MC; ++m) {
                    const int c = lane + 32 * m;
                    float v = 0.f;
                    if (arow && (cb[m] & 3)) {
                        const int b = (cb[m] >> 2) - 1;
                        const float tb = ctb[m];
                        float s0 = 0.f, s1 = 0.f;
                        if (cb[m] & 1) s0 = wa0 * __ldg(pc0 + b) + wa1 * __ldg(pc1 + b);
                        if (cb[m] & 2) s1 = wa0 * __ldg(pc0 + b + 1) + wa1 * __ldg(pc1 + b + 1);
                        v = m2 * ((1.f - tb) * s0 + tb * s1);
                    }
                    if (c < pitch) trow[swz_col(c)] = v;
                }
            }
        } else {
            // S7: G_b(i,j,k) = sum over the patient voxels (x,y) of slice z = j whose bilinear stencil reaches
            // beam voxel (i,k), weight (1-|du|)(1-|dw|), times g — the exact transpose of k_gather_dose.
            const float hx = (fabsf(d.cg) * P.du + fabsf(d.sg) * P.dw) / P.sx, hy = (fabsf(d.sg) * P.du + fabsf(d.cg) * P.dw) / P.sy;
            const float fu_x = d.cg * P.sx / P.du, fu_y = d.sg * P.sy / P.du, fw_x = -d.sg * P.sx / P.dw, fw_y = d.cg * P.sy / P.dw;
            const float w = P.wmin + k * P.dw;
            for (int r = warp; r < rows; r += CONV_THREADS / 32) {
                const int i = tu0 + r;
                float *trow = tile + r * pitch;
                float acc[MC];
#pragma unroll
                for (int m = 0; m < MC; ++m) acc[m] = 0.f;
                if (i >= 0 && i < P.Nu) {
                    const float u = (i - P.cu) * P.du;
                    const float fx = (P.isox + u * d.cg - w * d.sg - P.ox) / P.sx;
                    const float fy = (P.isoy + u * d.sg + w * d.cg - P.oy) / P.sy;
                    const int xa = max(0, (int)ceilf(fx - hx)), xb = min(P.nx - 1, (int)floorf(fx + hx));
                    const int ya = max(0, (int)ceilf(fy - hy)), yb = min(P.ny - 1, (int)floorf(fy + hy));
                    const float dxa = P.ox + xa * P.sx - P.isox, dya = P.oy + ya * P.sy - P.isoy;
                    const float eu0 = (d.cg * dxa + d.sg * dya) / P.du + P.cu - (float)i;
                    const float ew0 = (-d.sg * dxa + d.cg * dya - P.wmin) / P.dw - (float)k;
                    if (xb - xa <= 2 && yb - ya <= 2) {
                        // usual case (beam spacing ~ patient spacing): at most 3 x 3 candidates; all weights first,
                        // then all loads of a column batched so that their latencies overlap
                        float wg[9];
#pragma unroll
                        for (int cy = 0; cy < 3; ++cy)
#pragma unroll
                            for (int cx = 0; cx < 3; ++cx) {
                                const float wu = 1.f - fabsf(eu0 + cy * fu_y + cx * fu_x), ww = 1.f - fabsf(ew0 + cy * fw_y + cx * fw_x);
                                wg[cy * 3 + cx] = (wu > 0.f && ww > 0.f && xa + cx <= xb && ya + cy <= yb) ? wu * ww : 0.f;
                            }
                        const float *g0 = gT + ((size_t)ya * P.nx + xa) * P.nz;
#pragma unroll
                        for (int m = 0; m < MC; ++m) {
                            const int j = tv0 + lane + 32 * m;
                            const bool jin = lane + 32 * m < pitch && j >= 0 && j < P.Nv;
                            float v[9];
#pragma unroll
                            for (int cy = 0; cy < 3; ++cy)
#pragma unroll
                                for (int cx = 0; cx < 3; ++cx)
                                    v[cy * 3 + cx] = (jin && wg[cy * 3 + cx] != 0.f) ? __ldg(g0 + ((size_t)cy * P.nx + cx) * P.nz + j) : 0.f;
#pragma unroll
                            for (int q = 0; q < 9; ++q) acc[m] = fmaf(wg[q], v[q], acc[m]);
                        }
                    } else {
                        for (int yy = ya; yy <= yb; ++yy) {
                            const float euy = eu0 + (yy - ya) * fu_y, ewy = ew0 + (yy - ya) * fw_y;
                            for (int xx = xa; xx <= xb; ++xx) {
                                const float wu = 1.f - fabsf(euy + (xx - xa) * fu_x), ww = 1.f - fabsf(ewy + (xx - xa) * fw_x);
                                if (wu > 0.f && ww > 0.f) {           // warp-uniform
                                    const float wgt = wu * ww;
                                    const float *gcol = gT + ((size_t)yy * P.nx + xx) * P.nz;
#pragma unroll
                                    for (int m = 0; m < MC; ++m) {
                                        const int j = tv0 + lane + 32 * m;
                                        if (lane + 32 * m < pitch && j >= 0 && j < P.Nv) acc[m] = fmaf(wgt, __ldg(gcol + j), acc[m]);
                                    }
                                }
                            }
                        }
                    }
                }
#pragma unroll
                for (int m = 0; m < MC; ++m) {
                    const int c = lane + 32 * m;
                    if (c < pitch) trow[swz_col(c)] = acc[m];
                }
            }
        }
        __syncthreads();

        for (int t = tid; t < naf * nas; t += CONV_THREADS) {
            const int ts = t / naf, tf = t - ts * naf;
            float acc[RS][RF];
#pragma unroll
            for (int ii = 0; ii < RS; ++ii)
#pragma unroll
                for (int r = 0; r < RF; ++r) acc[ii][r] = 0.f;
            // forward: tile rows outside S_k hold zeros (structurally zero fluence) and are skipped
            const int ylo = ADJ ? 0 : max(0, S.u0 - tu0 - ts * RS), yhi = ADJ ? KT + RS - 2 : min(KT + RS - 2, S.u1 - tu0 - ts * RS);
            const float *xrow = tile + (ts * RS + ylo) * pitch;
            int xoff[NXQ];
#pragma unroll
            for (int q = 0; q < NXQ; ++q) xoff[q] = swz_col(tf * RF + 4 * q);
#pragma unroll 1
            for (int y = ylo; y <= yhi; ++y) {
                float x[XW];
#pragma unroll
                for (int q = 0; q < NXQ; ++q) {
                    const float4 v = *reinterpret_cast<const float4 *>(xrow + xoff[q]);
                    x[4 * q] = v.x; x[4 * q + 1] = v.y; x[4 * q + 2] = v.z; x[4 * q + 3] = v.w;
                }
#pragma unroll
                for (int ii = 0; ii < RS; ++ii) {
                    const int di = y - ii;
                    if (di >= 0 && di < KT) {
                        const float4 *w4 = reinterpret_cast<const float4 *>(Ws + di * KP);
#pragma unroll
                        for (int q = 0; q < KP / 4; ++q) {
                            const float4 wv = w4[q];
                            const float wq[4] = { wv.x, wv.y, wv.z, wv.w };
#pragma unroll
                            for (int e = 0; e < 4; ++e) {
                                const int dj = 4 * q + e;
                                if (dj < KT) {
#pragma unroll
                                    for (int r = 0; r < RF; ++r) acc[ii][r] = fmaf(wq[e], x[r + dj], acc[ii][r]);
                                }
                            }
                        }
                    }
                }
                xrow += pitch;
            }
#pragma unroll
            for (int ii = 0; ii < RS; ++ii) {
                float4 *o = reinterpret_cast<float4 *>(oslice + (size_t)((ats0 + ts) * RS + ii) * d.pv + (atf0 + tf) * RF);
                o[0] = make_float4(acc[ii][0], acc[ii][1], acc[ii][2], acc[ii][3]);
                o[1] = make_float4(acc[ii][4], acc[ii][5], acc[ii][6], acc[ii][7]);
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

// dL/dDose [nz][ny][nx] -> gT [ny*nx][nz] (z fastest), 32x32 shared-memory tiles.  Grid: (ceil(nxy/32), ceil(nz/32)).
__global__ void __launch_bounds__(256) k_transpose_g(int nxy, int nz, const float *__restrict__ g, float *__restrict__ gT)
{
    __shared__ float t[32][33];
    const int p0 = blockIdx.x * 32, z0 = blockIdx.y * 32;
    const int lx = threadIdx.x & 31, ly = threadIdx.x >> 5;
    for (int r = ly; r < 32; r += 8) {
        const int z = z0 + r, p = p0 + lx;
        t[r][lx] = (z < nz && p < nxy) ? __ldg(g + (size_t)z * nxy + p) : 0.f;
    }
    __syncthreads();
    for (int r = ly; r < 32; r += 8) {
        const int p = p0 + r, z = z0 + lx;
        if (p < nxy && z < nz) gT[(size_t)p * nz + z] = t[lx][r];
    }
}

}  // namespace pdrt
