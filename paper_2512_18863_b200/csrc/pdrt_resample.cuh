// pdrt_resample.cuh — S6 (beam -> patient resampling + MU-weighted accumulation, PAPER.md:160-168,
// Eq. 9) and S9 (transpose of the divergent projection, Eq. 5-6, in gather form).  These are the
// bandwidth-bound stages: each patient voxel is written once per call (accumulation over control points
// stays in registers), the compact D_b blocks are read once as 16-byte vectors along v, and no global
// atomics are used anywhere.  (S7, the transpose of S6, is k_resample_adjoint in pdrt_conv.cuh.)
#pragma once
#include "pdrt_dev.cuh"

namespace pdrt {

constexpr int GATHER_TX = 16, GATHER_TY = 4;   // block = 16 x 4 patient columns (x,y): two warp patches of 8 x 4 ...
constexpr int GATHER_Z = 32;            // ... times 32 z-slices
constexpr int GATHER_SPLIT = 4;         // ... times 4 warps per patch that share the control-point list round-robin
constexpr int GATHER_THREADS = 2 * GATHER_SPLIT * 32;
constexpr int GATHER_CHUNK = 128;       // control points staged in shared memory per pass

struct GatherCp {                       // the slice of CpDesc the resampler needs
    float cg, sg, scale;
    int ri0, pu, rj0, pv;
    int pad_;
    long long base;                     // slot * stride_cp
};

// S6.  Grid: (ceil(nx/16), ceil(ny/4), ceil(nz/32)); a block owns 16 x 4 patient columns (x,y) times 32
// z-slices, a warp an 8(x) x 4(y) patch of columns (compact in the beam frame under any gantry rotation).
//   dose[p] (+)= sum_b scale_b * bilinear_0(D_b[.][z][.]; fu, fw)
// The gantry rotates about z (G1), so for one control point the beam-frame position (fu, fw) and the
// four bilinear weights of a column are the same for all its voxels.  Per control point each lane computes
// them for ONE of the warp's 32 columns; the warp then walks the columns four at a time with 8 lanes along v
// per column, taking offset and weights by warp shuffle: every load instruction reads four full 128-byte
// lines of the v-fastest D_b block.  A lane accumulates 8 column groups x 4 z in registers over all control
// points (in control-point order: deterministic) and every patient voxel is written exactly once.
// Warp 0 first compacts the control points whose compact region can intersect this block.  The per-control-point
// chain (setup -> shuffle -> load -> accumulate) is latency-bound, so four warps share the list of one patch
// (entries q = s, s+4, ...) and their partial sums are added through shared memory in a fixed order.
__global__ void __launch_bounds__(GATHER_THREADS)
k_gather_dose(Params P, const CpDesc *__restrict__ desc, int cp0, int n_cp, const float *__restrict__ D,
              float *__restrict__ dose, int accumulate)
{
    __shared__ GatherCp list[GATHER_CHUNK];
    __shared__ int n_list;
    __shared__ float4 part[2 * (GATHER_SPLIT - 1)][8][32];
    const int tid = threadIdx.x;
    const int wrp = tid >> 5, lane = tid & 31;
    const int patch = wrp & 1, split = wrp >> 1;
    const int px0 = blockIdx.x * GATHER_TX + patch * 8, py0 = blockIdx.y * GATHER_TY;
    const int z0 = blockIdx.z * GATHER_Z;
    // the column this lane sets up
    const int ix = px0 + (lane & 7), iy = py0 + (lane >> 3);
    const float dx = P.ox + ix * P.sx - P.isox, dy = P.oy + iy * P.sy - P.isoy;
    const bool inside = ix < P.nx && iy < P.ny;
    // tile corners (for culling), relative to the isocentre
    const float cx0 = P.ox + (blockIdx.x * GATHER_TX) * P.sx - P.isox, cx1 = cx0 + (GATHER_TX - 1) * P.sx;
    const float cy0 = P.oy + (blockIdx.y * GATHER_TY) * P.sy - P.isoy, cy1 = cy0 + (GATHER_TY - 1) * P.sy;
    const int sub = lane >> 3, zl = 4 * (lane & 7);      // column within a group of four, z offset of this lane's quad
    float4 acc[8];
#pragma unroll
    for (int g = 0; g < 8; ++g) acc[g] = make_float4(0.f, 0.f, 0.f, 0.f);

    for (int c0 = 0; c0 < n_cp; c0 += GATHER_CHUNK) {
        __syncthreads();
        if (tid < 32) {                 // warp 0 builds the ordered list of candidate control points
            int count = 0;
            const int cend = min(n_cp, c0 + GATHER_CHUNK);
            for (int cb = c0; cb < cend; cb += 32) {
                const int c = cb + tid;
                bool keep = false;
                CpDesc d;
                if (c < cend) {
                    d = desc[cp0 + c];
                    if (d.a0 <= d.a1 && z0 < d.rj0 + d.pv && z0 + GATHER_Z > d.rj0) {
                        // u-extent of the tile: extremes are at its corners
                        const float u00 = d.cg * cx0 + d.sg * cy0, u10 = d.cg * cx1 + d.sg * cy0;
                        const float u01 = d.cg * cx0 + d.sg * cy1, u11 = d.cg * cx1 + d.sg * cy1;
                        const float umin = fminf(fminf(u00, u10), fminf(u01, u11)) / P.du + P.cu;
                        const float umax = fmaxf(fmaxf(u00, u10), fmaxf(u01, u11)) / P.du + P.cu;
                        keep = umax >= (float)(d.ri0 - 1) && umin <= (float)(d.ri0 + d.pu);
                    }
                }
                const unsigned m = __ballot_sync(0xffffffffu, keep);
                if (keep) {
                    GatherCp g;
                    g.cg = d.cg; g.sg = d.sg; g.scale = d.scale;
                    g.ri0 = d.ri0; g.pu = d.pu; g.rj0 = d.rj0; g.pv = d.pv; g.pad_ = 0;
                    g.base = (long long)c * P.stride_cp;
                    list[count + __popc(m & ((1u << tid) - 1u))] = g;
                }
                count += __popc(m);
            }
            if (tid == 0) n_list = count;
        }
        __syncthreads();
        const int n = n_list;
        for (int q = split; q < n; q += GATHER_SPLIT) {
            const GatherCp g = list[q];
            const float fu = (g.cg * dx + g.sg * dy) / P.du + P.cu;
            const float fw = (-g.sg * dx + g.cg * dy - P.wmin) / P.dw;
            const float flu = floorf(fu), flw = floorf(fw);
            const int i0 = (int)flu, k0 = (int)flw;
            const float tu = fu - flu, tw = fw - flw;
            // bilinear_0: neighbours outside the beam grid contribute 0; outside the compact region D_b is 0
            const int ihi = min(P.Nu, g.ri0 + g.pu);
            const bool iv0 = i0 >= g.ri0 && i0 < ihi, iv1 = i0 + 1 >= g.ri0 && i0 + 1 < ihi;
            const bool kv0 = k0 >= 0 && k0 < P.Nw, kv1 = k0 + 1 >= 0 && k0 + 1 < P.Nw;
            const bool any = inside && (iv0 || iv1) && (kv0 || kv1);
            if (!__any_sync(0xffffffffu, any)) continue;
            // invalid neighbours get weight 0 and are folded onto the valid one, so that every address is readable
            const int ia = iv0 ? i0 : i0 + 1, ka = kv0 ? k0 : k0 + 1;
            const float wu0 = iv0 ? 1.f - tu : 0.f, wu1 = iv1 ? tu : 0.f, wk0 = kv0 ? 1.f - tw : 0.f, wk1 = kv1 ? tw : 0.f;
            int offp = 0;
            if (any) offp = ((ka * g.pu + (ia - g.ri0)) * g.pv) | ((iv0 && iv1) ? 1 : 0) | ((kv0 && kv1) ? 2 : 0) | 4;   // pv % 8 == 0
            const float w00 = g.scale * (wu0 * wk0), w10 = g.scale * (wu1 * wk0), w01 = g.scale * (wu0 * wk1), w11 = g.scale * (wu1 * wk1);
            const int zq = z0 - g.rj0 + zl;                              // multiple of 4
            const bool zok = zq >= 0 && zq + 4 <= g.pv;
            const float *Dc = D + g.base + zq;
            const int sk = g.pu * g.pv;
#pragma unroll
            for (int gq = 0; gq < 8; ++gq) {
                const int src = 4 * gq + sub;
                const int o = __shfl_sync(0xffffffffu, offp, src);
                const float f00 = __shfl_sync(0xffffffffu, w00, src), f10 = __shfl_sync(0xffffffffu, w10, src);
                const float f01 = __shfl_sync(0xffffffffu, w01, src), f11 = __shfl_sync(0xffffffffu, w11, src);
                if ((o & 4) && zok) {
                    const float *p = Dc + (o & ~7);
                    const int di = (o & 1) ? g.pv : 0, dk = (o & 2) ? sk : 0;
                    const float4 a = __ldg(reinterpret_cast<const float4 *>(p));
                    const float4 b = __ldg(reinterpret_cast<const float4 *>(p + di));
                    const float4 c = __ldg(reinterpret_cast<const float4 *>(p + dk));
                    const float4 e = __ldg(reinterpret_cast<const float4 *>(p + dk + di));
                    acc[gq].x += f00 * a.x + f10 * b.x + f01 * c.x + f11 * e.x;
                    acc[gq].y += f00 * a.y + f10 * b.y + f01 * c.y + f11 * e.y;
                    acc[gq].z += f00 * a.z + f10 * b.z + f01 * c.z + f11 * e.z;
                    acc[gq].w += f00 * a.w + f10 * b.w + f01 * c.w + f11 * e.w;
                }
            }
        }
    }
    // partial sums of the four warps of a patch, added in a fixed order
    __syncthreads();
    if (split > 0) {
#pragma unroll
        for (int gq = 0; gq < 8; ++gq) part[(split - 1) * 2 + patch][gq][lane] = acc[gq];
    }
    __syncthreads();
    if (split > 0) return;
#pragma unroll
    for (int gq = 0; gq < 8; ++gq) {
#pragma unroll
        for (int sp = 0; sp < GATHER_SPLIT - 1; ++sp) {
            const float4 v = part[sp * 2 + patch][gq][lane];
            acc[gq].x += v.x; acc[gq].y += v.y; acc[gq].z += v.z; acc[gq].w += v.w;
        }
    }
#pragma unroll
    for (int gq = 0; gq < 8; ++gq) {
        const int col = 4 * gq + sub;
        const int ox = px0 + (col & 7), oy = py0 + (col >> 3);
        if (ox >= P.nx || oy >= P.ny) continue;
        const float v[4] = { acc[gq].x, acc[gq].y, acc[gq].z, acc[gq].w };
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int iz = z0 + zl + e;
            if (iz < P.nz) {
                float *o = dose + ((size_t)iz * P.ny + oy) * P.nx + ox;
                *o = accumulate ? *o + v[e] : v[e];
            }
        }
    }
}

// S9.  gPhimap_b[pix] = sum_k mag_k^2 sum_{voxels} weight(voxel -> pix) * H_b[voxel]  in gather form.  The bilinear
// weight is separable, weight = wa(i; a, k) * wb(j; b, k), so a warp owns a tile of 8 (a) x 32 (b, lanes: the
// contiguous axis of H_b) pixels of the fluence support bbox and, per slice, walks the few voxel rows i that reach
// its 8 pixel columns: each lane contracts its (at most 4) voxels along v once per row, t = sum_j wb H[k][i][j]
// (coalesced), and adds wa * t to the pixels a that row reaches.  Grid: (ceil(Nuf/8) * ceil(Nvf/32), n_cp); the
// 8 warps of a block take the slices k = warp, warp + 8, ... of the same tile and are reduced through shared
// memory in a fixed order (deterministic, no atomics).
struct SliceGeo { float mag, su, sv, iu, iv; int u0, u1, v0, v1; };   // su = mag*du/Du, iu = Du/(mag*du)

constexpr int PROJ_THREADS = 256, PROJ_KG = PROJ_THREADS / 32, PROJ_A = 8, PROJ_TAPS = 4;

__global__ void __launch_bounds__(PROJ_THREADS)
k_project_adjoint(Params P, const CpDesc *__restrict__ desc, int cp0, int n_cp, const float *__restrict__ H,
                  float *__restrict__ gphimap)
{
    extern __shared__ float4 proj_smem4[];
    SliceGeo *geo = reinterpret_cast<SliceGeo *>(proj_smem4);
    __shared__ float red[PROJ_KG][PROJ_A][32];
    const int slot = blockIdx.y;
    if (slot >= n_cp) return;
    const int cp = cp0 + slot;
    const CpDesc d = desc[cp];
    if (d.a0 > d.a1) return;
    const int nag = (P.Nuf + PROJ_A - 1) / PROJ_A;
    const int ag = blockIdx.x % nag, bg = blockIdx.x / nag;
    const int A0 = d.a0 + ag * PROJ_A, B0 = d.b0 + bg * 32;
    if (A0 > d.a1 || B0 > d.b1) return;
    const int A1 = min(d.a1, A0 + PROJ_A - 1);
    const int tid = threadIdx.x, lane = tid & 31, kg = tid >> 5;
    for (int k = tid; k < P.Nw; k += PROJ_THREADS) {
        const SliceBox S = slice_support(P, d, k);
        const float dist = P.sid + P.wmin + k * P.dw, mag = P.sid / dist;
        SliceGeo q;
        q.mag = mag; q.su = mag * P.du / P.Du; q.sv = mag * P.dv / P.Dv;
        q.iu = P.Du / (mag * P.du); q.iv = P.Dv / (mag * P.dv);
        q.u0 = S.u0; q.u1 = S.u1; q.v0 = S.v0; q.v1 = S.v1;
        geo[k] = q;
    }
    __syncthreads();
    const int b = B0 + lane;
    const bool live = b <= d.b1;
    const float *Hc = H + (size_t)slot * (size_t)P.stride_cp;
    const float vb = P.v0 / P.dv;                       // v_j / dv = vb + j
    float acc[PROJ_A];
#pragma unroll
    for (int q = 0; q < PROJ_A; ++q) acc[q] = 0.f;
    for (int k = kg; k < P.Nw; k += PROJ_KG) {
        const SliceGeo q = geo[k];
        if (q.u0 > q.u1 || q.v0 > q.v1) continue;
        // voxels with fa(i) in (A0-1, A1+1):  i - cu in ((A0-1-cuf) iu, (A1+1-cuf) iu)
        const int ilo = max(q.u0, (int)floorf((A0 - 1 - P.cuf) * q.iu + P.cu)), ihi = min(q.u1, (int)ceilf((A1 + 1 - P.cuf) * q.iu + P.cu));
        int jlo = max(q.v0, (int)floorf((b - 1 - P.cvf) * q.iv - vb)), jhi = min(q.v1, (int)ceilf((b + 1 - P.cvf) * q.iv - vb));
        if (!live) jhi = jlo - 1;
        const float m2 = q.mag * q.mag;
        // v weights of this lane's (at most PROJ_TAPS) voxels, once per slice; wider stencils (beam voxels much finer than the
        // map pixels) take the general loop
        const bool few = __all_sync(0xffffffffu, jhi - jlo < PROJ_TAPS);
        float wbq[PROJ_TAPS];
#pragma unroll
        for (int e = 0; e < PROJ_TAPS; ++e) {
            const float wb = 1.f - fabsf((vb + jlo + e) * q.sv + P.cvf - (float)b);
            wbq[e] = (jlo + e <= jhi && wb > 0.f) ? wb : 0.f;
        }
        for (int i = ilo; i <= ihi; ++i) {
            const float *hrow = Hc + ((size_t)k * d.pu + (i - d.ri0)) * d.pv - d.rj0;
            float t = 0.f;
            if (few) {
                float hv[PROJ_TAPS];
#pragma unroll
                for (int e = 0; e < PROJ_TAPS; ++e) hv[e] = wbq[e] != 0.f ? __ldg(hrow + jlo + e) : 0.f;
#pragma unroll
                for (int e = 0; e < PROJ_TAPS; ++e) t = fmaf(wbq[e], hv[e], t);
            } else {
                for (int j = jlo; j <= jhi; ++j) {
                    const float wb = 1.f - fabsf((vb + j) * q.sv + P.cvf - (float)b);
                    if (wb > 0.f) t = fmaf(wb, __ldg(hrow + j), t);
                }
            }
            t *= m2;
            const float fa = (i - P.cu) * q.su + P.cuf - (float)A0;      // uniform across the warp
#pragma unroll
            for (int e = 0; e < PROJ_A; ++e) {
                const float wa = 1.f - fabsf(fa - (float)e);
                if (wa > 0.f) acc[e] = fmaf(wa, t, acc[e]);
            }
        }
    }
#pragma unroll
    for (int e = 0; e < PROJ_A; ++e) red[kg][e][lane] = acc[e];
    __syncthreads();
    {
        const int e = tid >> 5;                          // PROJ_A == PROJ_KG: thread (e, lane) sums one pixel
        float s = 0.f;
#pragma unroll
        for (int q = 0; q < PROJ_KG; ++q) s += red[q][e][lane];
        if (live && A0 + e <= A1) gphimap[((size_t)cp * P.Nvf + b) * P.Nuf + A0 + e] = s;
    }
}

}  // namespace pdrt
