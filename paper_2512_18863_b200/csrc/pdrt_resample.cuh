// pdrt_resample.cuh — S6 (beam -> patient resampling + MU-weighted accumulation, PAPER.md:160-168,
// Eq. 9), S7 (its exact transpose in gather form) and S9 (transpose of the divergent projection,
// Eq. 5-6, in gather form).  These are the bandwidth-bound stages: each patient voxel is written once
// per call (accumulation over control points stays in a register), the compact D_b blocks are read
// once, and no global atomics are used anywhere.
#pragma once
#include "pdrt_dev.cuh"

namespace pdrt {

constexpr int GATHER_TX = 32, GATHER_TY = 8, GATHER_THREADS = GATHER_TX * GATHER_TY;
constexpr int GATHER_CHUNK = 128;       // control points staged in shared memory per pass

struct GatherCp {                       // the slice of CpDesc the resampler needs
    float cg, sg, scale;
    int ri0, pu, rj0;
    long long base;                     // slot*stride_cp - rj0*Nw*pu - ri0  (so index = base + (j*Nw + k)*pu + i)
};

// S6.  Grid: (ceil(nx/32), ceil(ny/8), nz); block 32x8 patient voxels of one z-slice.
// dose[p] (+)= sum_b scale_b * bilinear_0(D_b[.][z][.]; fu, fw).  A warp first compacts, in control-point
// order (deterministic summation), the control points whose compact region can intersect this tile.
__global__ void __launch_bounds__(GATHER_THREADS)
k_gather_dose(Params P, const CpDesc *__restrict__ desc, int cp0, int n_cp, const float *__restrict__ D,
              float *__restrict__ dose, int accumulate)
{
    __shared__ GatherCp list[GATHER_CHUNK];
    __shared__ int n_list;
    // each warp covers an 8(x) x 4(y) patch, so that under any gantry rotation its 32 voxels land in a compact
    // patch of the beam frame (a handful of 32-byte sectors per load instead of up to 32)
    const int tid = threadIdx.y * GATHER_TX + threadIdx.x;
    const int wrp = tid >> 5, lane = tid & 31;
    const int tx = (wrp & 3) * 8 + (lane & 7), ty = (wrp >> 2) * 4 + (lane >> 3);
    const int ix = blockIdx.x * GATHER_TX + tx, iy = blockIdx.y * GATHER_TY + ty, iz = blockIdx.z;
    const float dx = P.ox + ix * P.sx - P.isox, dy = P.oy + iy * P.sy - P.isoy;
    // tile corners (for culling), relative to the isocentre
    const float cx0 = P.ox + (blockIdx.x * GATHER_TX) * P.sx - P.isox, cx1 = cx0 + (GATHER_TX - 1) * P.sx;
    const float cy0 = P.oy + (blockIdx.y * GATHER_TY) * P.sy - P.isoy, cy1 = cy0 + (GATHER_TY - 1) * P.sy;
    const bool inside = ix < P.nx && iy < P.ny;
    float acc = 0.f;

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
                    if (d.a0 <= d.a1 && iz >= d.rj0 && iz < d.rj0 + d.pv) {
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
                    g.ri0 = d.ri0; g.pu = d.pu; g.rj0 = d.rj0;
                    g.base = (long long)c * P.stride_cp - ((long long)d.rj0 * P.Nw) * d.pu - d.ri0;
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
            const float *p = D + g.base + ((long long)iz * P.Nw + k0) * g.pu + i0;
            float s = 0.f;
            if (kv0) {
                if (iv0) s += (1.f - tu) * (1.f - tw) * __ldg(p);
                if (iv1) s += tu * (1.f - tw) * __ldg(p + 1);
            }
            if (kv1) {
                if (iv0) s += (1.f - tu) * tw * __ldg(p + g.pu);
                if (iv1) s += tu * tw * __ldg(p + g.pu + 1);
            }
            acc = fmaf(g.scale, s, acc);
        }
    }
    if (inside) {
        float *o = dose + ((size_t)iz * P.ny + iy) * P.nx + ix;
        *o = accumulate ? *o + acc : acc;
    }
}

// S7.  G_b = R_b^T g in gather form: for every beam voxel of the compact region, the patient voxels of the
// same z-slice whose bilinear stencil (as evaluated by k_gather_dose) reaches it.  Grid: (X, n_cp); each warp
// strides over 8(u) x 4(w) patches of the region (compact in the patient frame under any rotation) and writes
// the whole region (zeros outside the beam grid) so the conv adjoint can tile freely.
__global__ void __launch_bounds__(256)
k_resample_adjoint(Params P, const CpDesc *__restrict__ desc, int cp0, int n_cp, const float *__restrict__ g,
                   float *__restrict__ G)
{
    const int slot = blockIdx.y;
    if (slot >= n_cp) return;
    const CpDesc d = desc[cp0 + slot];
    if (d.a0 > d.a1) return;
    const int lane = threadIdx.x & 31, li = lane & 7, lk = lane >> 3;
    const int nti = d.pu >> 3, ntk = (P.Nw + 3) >> 2;
    const long long n_tiles = (long long)d.pv * ntk * nti;
    const long long warp0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5, n_warps = ((long long)gridDim.x * blockDim.x) >> 5;
    // half-extent, in patient indices, of the rotated unit hat of one beam voxel
    const float hx = (fabsf(d.cg) * P.du + fabsf(d.sg) * P.dw) / P.sx, hy = (fabsf(d.sg) * P.du + fabsf(d.cg) * P.dw) / P.sy;
    // beam-index increments per patient-index step
    const float fu_x = d.cg * P.sx / P.du, fu_y = d.sg * P.sy / P.du, fw_x = -d.sg * P.sx / P.dw, fw_y = d.cg * P.sy / P.dw;
    float *Gc = G + (size_t)slot * (size_t)P.stride_cp;
    for (long long wt = warp0; wt < n_tiles; wt += n_warps) {
        const int ti = (int)(wt % nti);
        const long long r = wt / nti;
        const int tk = (int)(r % ntk), jrel = (int)(r / ntk);
        const int i = d.ri0 + ti * 8 + li, k = tk * 4 + lk, j = d.rj0 + jrel;
        if (k >= P.Nw) continue;
        float acc = 0.f;
        if (i < P.Nu) {
            const float u = (i - P.cu) * P.du, w = P.wmin + k * P.dw;
            const float fx = (P.isox + u * d.cg - w * d.sg - P.ox) / P.sx;
            const float fy = (P.isoy + u * d.sg + w * d.cg - P.oy) / P.sy;
            const int xa = max(0, (int)ceilf(fx - hx)), xb = min(P.nx - 1, (int)floorf(fx + hx));
            const int ya = max(0, (int)ceilf(fy - hy)), yb = min(P.ny - 1, (int)floorf(fy + hy));
            const float *gz = g + (size_t)j * P.ny * P.nx;
            // beam-index offset of candidate (xa, ya) from this voxel, then incremental updates
            const float dxa = P.ox + xa * P.sx - P.isox, dya = P.oy + ya * P.sy - P.isoy;
            const float eu0 = (d.cg * dxa + d.sg * dya) / P.du + P.cu - (float)i;
            const float ew0 = (-d.sg * dxa + d.cg * dya - P.wmin) / P.dw - (float)k;
            for (int yy = ya; yy <= yb; ++yy) {
                const float euy = eu0 + (yy - ya) * fu_y, ewy = ew0 + (yy - ya) * fw_y;
                const float *grow = gz + (size_t)yy * P.nx;
                for (int xx = xa; xx <= xb; ++xx) {
                    const float wu = 1.f - fabsf(euy + (xx - xa) * fu_x), ww = 1.f - fabsf(ewy + (xx - xa) * fw_x);
                    if (wu > 0.f && ww > 0.f) acc = fmaf(wu * ww, __ldg(grow + xx), acc);
                }
            }
        }
        Gc[((size_t)jrel * P.Nw + k) * d.pu + (i - d.ri0)] = acc;
    }
}

// S9.  gPhimap_b[pix] = sum_k mag_k^2 sum_{voxels} weight(voxel -> pix) * H_b[voxel]  in gather form: for each
// pixel of the fluence support bbox and each slice, the (at most 3x3) voxels of S_k whose bilinear stencil
// reaches the pixel.  Grid: (ceil(Nuf*Nvf/32), n_cp); block 256 = 32 consecutive bbox pixels x 8 slice groups,
// per-slice geometry staged once in shared memory, slice groups reduced through shared memory.
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
    const int bw = d.a1 - d.a0 + 1, npx = bw * (d.b1 - d.b0 + 1);
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
    const int a = d.a0 + (live ? p % bw : 0), b = d.b0 + (live ? p / bw : 0);
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
            for (int j = jlo; j <= jhi; ++j) {
                const float wb = 1.f - fabsf((vb + j) * q.sv + P.cvf - (float)b);
                if (wb <= 0.f) continue;
                const float *hrow = Hc + ((size_t)(j - d.rj0) * P.Nw + k) * d.pu - d.ri0;
                for (int i = ilo; i <= ihi; ++i) {
                    const float wa = 1.f - fabsf((i - P.cu) * q.su + P.cuf - (float)a);
                    if (wa > 0.f) s = fmaf(wa * wb, __ldg(hrow + i), s);
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
