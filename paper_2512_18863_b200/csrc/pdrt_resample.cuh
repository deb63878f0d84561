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
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * GATHER_TX + tx;
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
// same z-slice whose bilinear stencil (as evaluated by k_gather_dose) reaches it.  Grid: (X, n_cp), grid-stride
// over the region; writes the whole region (zeros outside the beam grid) so the conv adjoint can tile freely.
__global__ void __launch_bounds__(256)
k_resample_adjoint(Params P, const CpDesc *__restrict__ desc, int cp0, int n_cp, const float *__restrict__ g,
                   float *__restrict__ G)
{
    const int slot = blockIdx.y;
    if (slot >= n_cp) return;
    const CpDesc d = desc[cp0 + slot];
    if (d.a0 > d.a1) return;
    const long long n = (long long)d.pu * d.pv * P.Nw;
    // half-extent, in patient indices, of the rotated unit hat of one beam voxel
    const float hx = (fabsf(d.cg) * P.du + fabsf(d.sg) * P.dw) / P.sx, hy = (fabsf(d.sg) * P.du + fabsf(d.cg) * P.dw) / P.sy;
    float *Gc = G + (size_t)slot * (size_t)P.stride_cp;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
        const int irel = (int)(e % d.pu);
        const long long r = e / d.pu;
        const int k = (int)(r % P.Nw), jrel = (int)(r / P.Nw);
        const int i = d.ri0 + irel, j = d.rj0 + jrel;
        float acc = 0.f;
        if (i < P.Nu) {
            const float u = (i - P.cu) * P.du, w = P.wmin + k * P.dw;
            const float fx = (P.isox + u * d.cg - w * d.sg - P.ox) / P.sx;
            const float fy = (P.isoy + u * d.sg + w * d.cg - P.oy) / P.sy;
            const int xa = max(0, (int)ceilf(fx - hx)), xb = min(P.nx - 1, (int)floorf(fx + hx));
            const int ya = max(0, (int)ceilf(fy - hy)), yb = min(P.ny - 1, (int)floorf(fy + hy));
            const float *gz = g + (size_t)j * P.ny * P.nx;
            for (int yy = ya; yy <= yb; ++yy) {
                const float dy = P.oy + yy * P.sy - P.isoy;
                for (int xx = xa; xx <= xb; ++xx) {
                    const float dx = P.ox + xx * P.sx - P.isox;
                    const float fu = (d.cg * dx + d.sg * dy) / P.du + P.cu;
                    const float fw = (-d.sg * dx + d.cg * dy - P.wmin) / P.dw;
                    const float wu = 1.f - fabsf(fu - (float)i), ww = 1.f - fabsf(fw - (float)k);
                    if (wu > 0.f && ww > 0.f) acc = fmaf(wu * ww, __ldg(gz + (size_t)yy * P.nx + xx), acc);
                }
            }
        }
        Gc[e] = acc;
    }
}

// S9.  gPhimap_b[pix] = sum_k mag_k^2 sum_{voxels} weight(voxel -> pix) * H_b[voxel]  in gather form: for each
// pixel of the fluence support bbox and each slice, the (at most 3x3) voxels of S_k whose bilinear stencil
// reaches the pixel.  Grid: (Nvf, n_cp); block 128 = 32 pixels x 4 slice groups, reduced through shared memory.
__global__ void __launch_bounds__(128)
k_project_adjoint(Params P, const CpDesc *__restrict__ desc, int cp0, int n_cp, const float *__restrict__ H,
                  float *__restrict__ gphimap)
{
    const int b = blockIdx.x, slot = blockIdx.y;
    if (slot >= n_cp) return;
    const int cp = cp0 + slot;
    const CpDesc d = desc[cp];
    if (d.a0 > d.a1 || b < d.b0 || b > d.b1) return;
    __shared__ float red[4][32];
    const int lane = threadIdx.x & 31, kg = threadIdx.x >> 5;
    const float *Hc = H + (size_t)slot * (size_t)P.stride_cp;
    float *out = gphimap + ((size_t)cp * P.Nvf + b) * P.Nuf;
    for (int a0 = d.a0; a0 <= d.a1; a0 += 32) {
        const int a = a0 + lane;
        float acc = 0.f;
        if (a <= d.a1) {
            for (int k = kg; k < P.Nw; k += 4) {
                const SliceBox S = slice_support(P, d, k);
                if (box_empty(S)) continue;
                const float dist = P.sid + P.wmin + k * P.dw, mag = P.sid / dist, inv_mag = dist / P.sid;
                const int ilo = max(S.u0, (int)floorf((a - 1 - P.cuf) * P.Du * inv_mag / P.du + P.cu));
                const int ihi = min(S.u1, (int)ceilf((a + 1 - P.cuf) * P.Du * inv_mag / P.du + P.cu));
                const int jlo = max(S.v0, (int)floorf(((b - 1 - P.cvf) * P.Dv * inv_mag - P.v0) / P.dv));
                const int jhi = min(S.v1, (int)ceilf(((b + 1 - P.cvf) * P.Dv * inv_mag - P.v0) / P.dv));
                float s = 0.f;
                for (int j = jlo; j <= jhi; ++j) {
                    const float fb = mag * (P.v0 + j * P.dv) / P.Dv + P.cvf;
                    const float wb = 1.f - fabsf(fb - (float)b);
                    if (wb <= 0.f) continue;
                    for (int i = ilo; i <= ihi; ++i) {
                        const float fa = mag * ((i - P.cu) * P.du) / P.Du + P.cuf;
                        const float wa = 1.f - fabsf(fa - (float)a);
                        if (wa > 0.f) s = fmaf(wa * wb, __ldg(Hc + ((size_t)(j - d.rj0) * P.Nw + k) * d.pu + (i - d.ri0)), s);
                    }
                }
                acc = fmaf(mag * mag, s, acc);
            }
        }
        red[kg][lane] = acc;
        __syncthreads();
        if (kg == 0 && a <= d.a1) out[a] = (red[0][lane] + red[1][lane]) + (red[2][lane] + red[3][lane]);
        __syncthreads();
    }
}

}  // namespace pdrt
