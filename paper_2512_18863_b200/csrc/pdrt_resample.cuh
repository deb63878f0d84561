// pdrt_resample.cuh — S6 (beam -> patient resampling + MU-weighted accumulation, PAPER.md:160-168,
// Eq. 9) and S9 (transpose of the divergent projection, Eq. 5-6, in gather form).  These are the
// bandwidth-bound stages: each patient voxel is written once per call (accumulation over control points
// stays in registers), the compact D_b blocks are read once as 16-byte vectors along v, and no global
// atomics are used anywhere.  (S7, the transpose of S6, lives in the tile fill of k_conv<K,true>.)
#pragma once
#include "pdrt_dev.cuh"

namespace pdrt {

constexpr int GATHER_T = 16;            // block = 16 x 16 patient columns (x,y) ...
constexpr int GATHER_Z = 16;            // ... times 16 z-slices per thread
constexpr int GATHER_THREADS = GATHER_T * GATHER_T;
constexpr int GATHER_CHUNK = 128;       // control points staged in shared memory per pass

struct GatherCp {                       // the slice of CpDesc the resampler needs
    float cg, sg, scale;
    int ri0, pu, rj0, pv;
    int pad_;
    long long base;                     // slot * stride_cp
};

// S6.  Grid: (ceil(nx/16), ceil(ny/16), ceil(nz/16)); each thread owns one patient column (x,y) and 16
// consecutive z-slices.  The gantry rotates about z (G1), so for one control point the beam-frame
// position (fu, fw) and the four bilinear weights are the same for all 16 voxels: they are computed once and
// the four neighbouring beam columns are streamed as float4 along v.
//   dose[p] (+)= sum_b scale_b * bilinear_0(D_b[.][z][.]; fu, fw)
// A warp first compacts, in control-point order (deterministic summation), the control points whose compact
// region can intersect this tile.  Each warp covers an 8(x) x 4(y) patch so that under any gantry rotation
// its 32 columns land in a compact patch of the beam frame.
__global__ void __launch_bounds__(GATHER_THREADS)
k_gather_dose(Params P, const CpDesc *__restrict__ desc, int cp0, int n_cp, const float *__restrict__ D,
              float *__restrict__ dose, int accumulate)
{
    __shared__ GatherCp list[GATHER_CHUNK];
    __shared__ int n_list;
    const int tid = threadIdx.x;
    const int wrp = tid >> 5, lane = tid & 31;
    const int tx = (wrp & 1) * 8 + (lane & 7), ty = (wrp >> 1) * 4 + (lane >> 3);
    const int ix = blockIdx.x * GATHER_T + tx, iy = blockIdx.y * GATHER_T + ty, z0 = blockIdx.z * GATHER_Z;
    const float dx = P.ox + ix * P.sx - P.isox, dy = P.oy + iy * P.sy - P.isoy;
    // tile corners (for culling), relative to the isocentre
    const float cx0 = P.ox + (blockIdx.x * GATHER_T) * P.sx - P.isox, cx1 = cx0 + (GATHER_T - 1) * P.sx;
    const float cy0 = P.oy + (blockIdx.y * GATHER_T) * P.sy - P.isoy, cy1 = cy0 + (GATHER_T - 1) * P.sy;
    const bool inside = ix < P.nx && iy < P.ny;
    float acc[GATHER_Z];
#pragma unroll
    for (int q = 0; q < GATHER_Z; ++q) acc[q] = 0.f;

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
        if (!inside) continue;
        const int n = n_list;
        for (int q = 0; q < n; ++q) {
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
            if (!(iv0 || iv1) || !(kv0 || kv1)) continue;
            const int zq0 = z0 - g.rj0;                              // multiple of 4 (rj0 % 4 == 0)
            const float *p = D + g.base + ((long long)k0 * g.pu + (i0 - g.ri0)) * g.pv + zq0;
            const long long sk = (long long)g.pu * g.pv;
            const float w00 = g.scale * ((1.f - tu) * (1.f - tw)), w10 = g.scale * (tu * (1.f - tw));
            const float w01 = g.scale * ((1.f - tu) * tw), w11 = g.scale * (tu * tw);
#pragma unroll
            for (int qd = 0; qd < GATHER_Z / 4; ++qd) {
                const int zq = zq0 + 4 * qd;
                if (zq < 0 || zq + 4 > g.pv) continue;               // uniform across the block
                float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a, c = a, e = a;
                if (kv0 && iv0) a = __ldg(reinterpret_cast<const float4 *>(p + 4 * qd));
                if (kv0 && iv1) b = __ldg(reinterpret_cast<const float4 *>(p + g.pv + 4 * qd));
                if (kv1 && iv0) c = __ldg(reinterpret_cast<const float4 *>(p + sk + 4 * qd));
                if (kv1 && iv1) e = __ldg(reinterpret_cast<const float4 *>(p + sk + g.pv + 4 * qd));
                acc[4 * qd + 0] += w00 * a.x + w10 * b.x + w01 * c.x + w11 * e.x;
                acc[4 * qd + 1] += w00 * a.y + w10 * b.y + w01 * c.y + w11 * e.y;
                acc[4 * qd + 2] += w00 * a.z + w10 * b.z + w01 * c.z + w11 * e.z;
                acc[4 * qd + 3] += w00 * a.w + w10 * b.w + w01 * c.w + w11 * e.w;
            }
        }
    }
    if (inside) {
#pragma unroll
        for (int q = 0; q < GATHER_Z; ++q) {
            const int iz = z0 + q;
            if (iz < P.nz) {
                float *o = dose + ((size_t)iz * P.ny + iy) * P.nx + ix;
                *o = accumulate ? *o + acc[q] : acc[q];
            }
        }
    }
}

// S9.  gPhimap_b[pix] = sum_k mag_k^2 sum_{voxels} weight(voxel -> pix) * H_b[voxel]  in gather form: for each
// pixel of the fluence support bbox and each slice, the (at most 3x3) voxels of S_k whose bilinear stencil
// reaches the pixel.  Grid: (ceil(Nuf*Nvf/32), n_cp); block 256 = 32 consecutive bbox pixels (running along v,
// the contiguous axis of H_b) x 8 slice groups, per-slice geometry staged once in shared memory, slice groups
// reduced through shared memory.
struct SliceGeo { float mag, su, sv, iu, iv; int u0, u1, v0, v1; };   // su = mag*du/Du, iu = Du/(mag*du)

constexpr int PROJ_THREADS = 256, PROJ_KG = PROJ_THREADS / 32;

__global__ void __launch_bounds__(PROJ_THREADS)
k_project_adjoint(Params P, const CpDesc *__restrict__ desc, int cp0, int n_cp, const float *__restrict__ H,
                  float *__restrict__ gphimap)
{
    extern __shared__ float4 proj_smem4[];
    SliceGeo *geo = reinterpret_cast<SliceGeo *>(proj_smem4);
    __shared__ float red[PROJ_KG][32];
    const int slot = blockIdx.y;
    if (slot >= n_cp) return;
    const int cp = cp0 + slot;
    const CpDesc d = desc[cp];
    if (d.a0 > d.a1) return;
    const int bh = d.b1 - d.b0 + 1, npx = bh * (d.a1 - d.a0 + 1);
    const int p0 = blockIdx.x * 32;
    if (p0 >= npx) return;
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
    const int p = p0 + lane;
    const bool live = p < npx;
    const int a = d.a0 + (live ? p / bh : 0), b = d.b0 + (live ? p % bh : 0);
    const float *Hc = H + (size_t)slot * (size_t)P.stride_cp;
    const float vb = P.v0 / P.dv;                       // v_j / dv = vb + j
    float acc = 0.f;
    if (live) {
        for (int k = kg; k < P.Nw; k += PROJ_KG) {
            const SliceGeo q = geo[k];
            if (q.u0 > q.u1 || q.v0 > q.v1) continue;
            // voxels with fa(i) in (a-1, a+1):  i - cu in ((a-1-cuf) iu, (a+1-cuf) iu)
            const int ilo = max(q.u0, (int)floorf((a - 1 - P.cuf) * q.iu + P.cu)), ihi = min(q.u1, (int)ceilf((a + 1 - P.cuf) * q.iu + P.cu));
            const int jlo = max(q.v0, (int)floorf((b - 1 - P.cvf) * q.iv - vb)), jhi = min(q.v1, (int)ceilf((b + 1 - P.cvf) * q.iv - vb));
            float s = 0.f;
            for (int i = ilo; i <= ihi; ++i) {
                const float wa = 1.f - fabsf((i - P.cu) * q.su + P.cuf - (float)a);
                if (wa <= 0.f) continue;
                const float *hrow = Hc + ((size_t)k * d.pu + (i - d.ri0)) * d.pv - d.rj0;
                for (int j = jlo; j <= jhi; ++j) {
                    const float wb = 1.f - fabsf((vb + j) * q.sv + P.cvf - (float)b);
                    if (wb > 0.f) s = fmaf(wa * wb, __ldg(hrow + j), s);
                }
            }
            acc = fmaf(q.mag * q.mag, s, acc);
        }
    }
    red[kg][lane] = acc;
    __syncthreads();
    if (kg == 0 && live) {
        float s = 0.f;
#pragma unroll
        for (int q = 0; q < PROJ_KG; ++q) s += red[q][lane];
        gphimap[((size_t)cp * P.Nvf + b) * P.Nuf + a] = s;
    }
}

}  // namespace pdrt
