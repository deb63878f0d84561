// pdrt_fluence.cuh — S1 aperture -> fluence rasteriser, the per-control-point descriptor, and S10
// (rasteriser adjoint + MU gradient).  One block per control point; everything is confined to the
// fluence support bbox (jaw opening dilated by the blur half-widths), so cost follows the field size.
//
// PAPER.md:103-119:  A = sum_i ov_v ov_u (Eq. 4), J = jaw mask, Phi0 = J (tau + (1-tau) A),
// Phi1 = G_v(jaw) G_u(mlc) Phi0, Phi2 = Phi1 + sum_q amp_q G_u G_v Phi0, Phimap = Phi2 * OAR(r).
#pragma once
#include "pdrt_dev.cuh"

namespace pdrt {

constexpr int FLU_THREADS = 256;
constexpr int FLU_MAX_ROWS = 1024;   // pixel rows of a jaw opening with a precomputed leaf range (wider maps scan all pairs)

__device__ __forceinline__ float flu_u(const Params &P, int a) { return (a - P.cuf) * P.Du; }
__device__ __forceinline__ float flu_v(const Params &P, int b) { return (b - P.cvf) * P.Dv; }

__device__ __forceinline__ float oar_factor(const FluTables &T, float r)
{
    if (T.n_oar <= 0) return 1.f;
    const float t = r / T.oar_dr;
    const int n0 = (int)floorf(t);
    if (n0 >= T.n_oar - 1) return T.oar[T.n_oar - 1];
    const float f = t - n0;
    return (1.f - f) * T.oar[n0] + f * T.oar[n0 + 1];
}

// value of a bbox-confined map at (a,b); zero outside the bbox (zero padding of the blurs)
__device__ __forceinline__ float at_bbox(const float *m, const Params &P, const CpDesc &d, int a, int b)
{
    return (a >= d.a0 && a <= d.a1 && b >= d.b0 && b <= d.b1) ? m[b * P.Nuf + a] : 0.f;
}

// 1-D zero-padded convolution of a bbox-confined map along u (axis 0) or v (axis 1) at pixel (a,b)
__device__ __forceinline__ float blur_at(const float *m, const Params &P, const CpDesc &d, int a, int b,
                                         int axis, int T, const float *g)
{
    float s = 0.f;
    for (int t = -T; t <= T; ++t) {
        const int aa = axis == 0 ? a + t : a, bb = axis == 1 ? b + t : b;
        s += g[t + T] * at_bbox(m, P, d, aa, bb);
    }
    return s;
}

// A bbox-confined map either in shared memory (pitch = bbox width, origin = bbox corner) or in its global scratch plane (pitch Nuf).
struct MapView {
    float *p; int pitch, oa, ob;
    __device__ __forceinline__ float &at(int a, int b) const { return p[(b - ob) * pitch + (a - oa)]; }
};
// value at (a,b); zero outside the box [a0,a1] x [b0,b1] (zero padding of the blurs)
__device__ __forceinline__ float view_at(const MapView &m, int a0, int a1, int b0, int b1, int a, int b)
{
    return (a >= a0 && a <= a1 && b >= b0 && b <= b1) ? m.at(a, b) : 0.f;
}
__device__ __forceinline__ float view_blur(const MapView &m, const CpDesc &d, int a, int b, int axis, int T, const float *g)
{
    float s = 0.f;
    for (int t = -T; t <= T; ++t) s += g[t + T] * view_at(m, d.a0, d.a1, d.b0, d.b1, axis == 0 ? a + t : a, axis == 1 ? b + t : b);
    return s;
}
constexpr int FLU_TILE = 3072;       // pixels of a support bbox that k_fluence keeps in shared memory (three planes)

// Builds CpDesc: gantry axes, jaw and support bboxes, compact region, conv chunking, work counters.
__device__ void build_desc(const Params &P, const float *jaws, float gantry_deg, float coll_deg, float mu, CpDesc &d)
{
    const double phi = (double)gantry_deg * 3.14159265358979323846 / 180.0;
    d.cg = (float)cos(phi);
    d.sg = (float)sin(phi);
    const double phc = (double)coll_deg * 3.14159265358979323846 / 180.0;
    d.cc = coll_deg == 0.f ? 1.f : (float)cos(phc);
    d.sc = coll_deg == 0.f ? 0.f : (float)sin(phc);
    d.scale = P.cal * mu;
    const float x1 = jaws[0], x2 = jaws[1], y1 = jaws[2], y2 = jaws[3];
    const float eu = -0.5f * P.Nuf * P.Du, ev = -0.5f * P.Nvf * P.Dv;     // left edge of pixel 0
    // pixel of d ov/d lo: e_a < lo <= e_{a+1}; pixel of d ov/d hi: e_a <= hi < e_{a+1}
    d.ja0 = max(0, (int)ceilf((x1 - eu) / P.Du) - 1);
    d.ja1 = min(P.Nuf - 1, (int)floorf((x2 - eu) / P.Du));
    d.jb0 = max(0, (int)ceilf((y1 - ev) / P.Dv) - 1);
    d.jb1 = min(P.Nvf - 1, (int)floorf((y2 - ev) / P.Dv));
    const bool empty = d.ja0 > d.ja1 || d.jb0 > d.jb1 || !(x1 <= x2) || !(y1 <= y2);
    d.a0 = max(0, d.ja0 - P.Tu_max); d.a1 = min(P.Nuf - 1, d.ja1 + P.Tu_max);
    d.b0 = max(0, d.jb0 - P.Tv_max); d.b1 = min(P.Nvf - 1, d.jb1 + P.Tv_max);
    d.ri0 = d.rj0 = d.pu = d.pv = d.ntf = d.nts = 0;
    d.ncf = d.ntfc = d.n_items = d.n_items_adj = 0;
    d.support_vox = d.footprint_vox = d.region_vox = d.macs_fwd = d.macs_adj = 0ull;
    d.pa0 = d.pb0 = 1; d.pa1 = d.pb1 = 0;
    if (empty) { d.a0 = d.ja0 = 1; d.a1 = d.ja1 = 0; d.b0 = d.jb0 = 1; d.b1 = d.jb1 = 0; return; }
    // support bbox in the projection frame: the collimator-frame box, grown by the one-pixel reach of the bilinear resampling,
    // rotated by R(phi_c) about the axis; identical when the angle is 0
    d.pa0 = d.a0; d.pa1 = d.a1; d.pb0 = d.b0; d.pb1 = d.b1;
    if (d.sc != 0.f || d.cc != 1.f) {
        float ulo = 1e30f, uhi = -1e30f, vlo = 1e30f, vhi = -1e30f;
        for (int q = 0; q < 4; ++q) {
            const float uc = ((q & 1 ? d.a1 + 1 : d.a0 - 1) - P.cuf) * P.Du, vc = ((q & 2 ? d.b1 + 1 : d.b0 - 1) - P.cvf) * P.Dv;
            const float ur = d.cc * uc - d.sc * vc, vr = d.sc * uc + d.cc * vc;
            ulo = fminf(ulo, ur); uhi = fmaxf(uhi, ur); vlo = fminf(vlo, vr); vhi = fmaxf(vhi, vr);
        }
        d.pa0 = max(0, (int)floorf(ulo / P.Du + P.cuf)); d.pa1 = min(P.Nuf - 1, (int)ceilf(uhi / P.Du + P.cuf));
        d.pb0 = max(0, (int)floorf(vlo / P.Dv + P.cvf)); d.pb1 = min(P.Nvf - 1, (int)ceilf(vhi / P.Dv + P.cvf));
        if (d.pa0 > d.pa1 || d.pb0 > d.pb1) { d.a0 = d.ja0 = d.pa0 = 1; d.a1 = d.ja1 = d.pa1 = 0; d.b0 = d.jb0 = d.pb0 = 1; d.b1 = d.jb1 = d.pb1 = 0; return; }
    }
    const int C = P.CH;
    const SliceBox s0 = slice_support(P, d, 0), s1 = slice_support(P, d, P.Nw - 1);
    const int u0 = max(0, min(s0.u0, s1.u0) - C), u1 = min(P.Nu - 1, max(s0.u1, s1.u1) + C);
    const int v0 = max(0, min(s0.v0, s1.v0) - C), v1 = min(P.Nv - 1, max(s0.v1, s1.v1) + C);
    if (u0 > u1 || v0 > v1) { d.a0 = d.ja0 = d.pa0 = 1; d.a1 = d.ja1 = d.pa1 = 0; d.b0 = d.jb0 = d.pb0 = 1; d.b1 = d.jb1 = d.pb1 = 0; return; }
    d.ri0 = u0;
    d.pu = ((u1 - u0 + 1) + RS - 1) / RS * RS;
    d.rj0 = v0 & ~7;
    d.pv = ((v1 - d.rj0 + 1) + RF - 1) / RF * RF;
    d.ntf = d.pv / RF;
    d.nts = d.pu / RS;
    d.ncf = (d.ntf + P.ntfc_max - 1) / P.ntfc_max;
    d.ntfc = (d.ntf + d.ncf - 1) / d.ncf;
    // conv work items: one per slice and chunk along v (the warp that takes an item walks its active thread-tiles)
    d.n_items = d.n_items_adj = P.Nw * d.ncf;
    d.region_vox = (unsigned long long)d.pu * d.pv * P.Nw;
}

// S1.  Grid: n_cp blocks.  Scratch maps P0, T1, T2, A are [n_cp][Nvf][Nuf]; phimapT is [n_cp][Nuf][Nvf].
__global__ void __launch_bounds__(FLU_THREADS)
k_fluence(Params P, FluTables T, int n_cp, const float *__restrict__ leaves, const float *__restrict__ jaws,
          const float *__restrict__ gantry_deg, const float *__restrict__ coll_deg, const float *__restrict__ mu, CpDesc *desc,
          SliceBox16 *sbox, SliceBox16 *wbox,
          float *P0, float *T1, float *T2, float *Abuf, float *phimap, float *phimapT)
{
    const int cp = blockIdx.x, tid = threadIdx.x;
    if (cp >= n_cp) return;
    __shared__ CpDesc d;
    __shared__ unsigned long long cnt[4];
    if (tid == 0) {
        build_desc(P, jaws + 4 * cp, gantry_deg ? gantry_deg[cp] : 0.f, coll_deg ? coll_deg[cp] : 0.f, mu ? mu[cp] : 0.f, d);
        cnt[0] = cnt[1] = cnt[2] = cnt[3] = 0ull;
    }
    __syncthreads();
    const bool empty = d.a0 > d.a1;
    if (!empty) {     // per-slice boxes for the resampling kernels, and work counters: |S_k|, |F_k|, thread-tiles
        const int C = P.CH, CB = (P.KT - 1) / 2, nbh = (P.NB - 1) / 2;
        unsigned long long sup = 0, fp = 0, tf = 0, ta = 0;
        for (int k = tid; k < P.Nw; k += FLU_THREADS) {
            const SliceBox s = slice_support(P, d, k), f = dilate(P, s, C);
            SliceBox16 sb = { 1, 0, 1, 0 }, wb = { 1, 0, 1, 0 };
            if (!box_empty(s)) {
                sb.u0 = (short)s.u0; sb.u1 = (short)s.u1; sb.v0 = (short)s.v0; sb.v1 = (short)s.v1;
                // thread-tiles of the forward conv that intersect F_k (conv_load_item), clipped to the beam grid
                wb.u0 = (short)(d.ri0 + (f.u0 - d.ri0) / RS * RS);
                wb.u1 = (short)min(P.Nu - 1, d.ri0 + min(d.nts - 1, (f.u1 - d.ri0) / RS) * RS + RS - 1);
                wb.v0 = (short)(d.rj0 + (f.v0 - d.rj0) / RF * RF);
                wb.v1 = (short)(d.rj0 + (f.v1 - d.rj0) / RF * RF + RF - 1);
                if (P.conv_sym && d.ncf == 1) {     // k_conv_sym / k_conv_fold start their 8- / 4-column tiles at the box (16-byte aligned), clipped to the region
                    const int tw = P.conv_sym == 2 ? 4 : RF;
                    wb.v0 = (short)(f.v0 & ~3);
                    wb.v1 = (short)min(wb.v0 + ((f.v1 - wb.v0) / tw + 1) * tw - 1, d.rj0 + d.pv - 1);
                }
            }
            sbox[(size_t)cp * P.Nw + k] = sb;
            wbox[(size_t)cp * P.Nw + k] = wb;
            if (box_empty(s)) continue;
            sup += (unsigned long long)(s.u1 - s.u0 + 1) * (s.v1 - s.v0 + 1);
            fp += (unsigned long long)(f.u1 - f.u0 + 1) * (f.v1 - f.v0 + 1);
            // thread-tiles that do multiply-adds: forward, per pass the tiles the shifted sub-kernel reaches inside F_k; adjoint, S_k in every pass
            for (int bi = -nbh; bi <= nbh; ++bi)
                for (int bj = -nbh; bj <= nbh; ++bj) {
                    const int u0 = max(f.u0, s.u0 - bi * P.KT - CB), u1 = min(f.u1, s.u1 - bi * P.KT + CB);
                    const int v0 = max(f.v0, s.v0 - bj * P.KT - CB), v1 = min(f.v1, s.v1 - bj * P.KT + CB);
                    if (u0 <= u1 && v0 <= v1)
                        tf += (unsigned long long)((u1 - d.ri0) / RS - (u0 - d.ri0) / RS + 1) * ((v1 - d.rj0) / RF - (v0 - d.rj0) / RF + 1);
                }
            ta += (unsigned long long)P.NB * P.NB * ((s.u1 - d.ri0) / RS - (s.u0 - d.ri0) / RS + 1) * ((s.v1 - d.rj0) / RF - (s.v0 - d.rj0) / RF + 1);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            sup += __shfl_xor_sync(0xffffffffu, sup, o); fp += __shfl_xor_sync(0xffffffffu, fp, o);
            tf += __shfl_xor_sync(0xffffffffu, tf, o); ta += __shfl_xor_sync(0xffffffffu, ta, o);
        }
        if ((tid & 31) == 0) { atomicAdd(&cnt[0], sup); atomicAdd(&cnt[1], fp); atomicAdd(&cnt[2], tf); atomicAdd(&cnt[3], ta); }
    }
    __syncthreads();
    if (tid == 0) {
        d.support_vox = cnt[0]; d.footprint_vox = cnt[1];
        // k_conv: KT^2 multiply-adds per output of an active thread-tile; k_conv_sym counts what it executes itself
        d.macs_fwd = P.conv_sym ? 0ull : cnt[2] * (unsigned long long)(RF * RS * P.KT * P.KT);
        d.macs_adj = P.conv_sym ? 0ull : cnt[3] * (unsigned long long)(RF * RS * P.KT * P.KT);
        desc[cp] = d;
    }
    if (empty) return;

    const size_t mo = (size_t)cp * P.Nuf * P.Nvf;
    float *Am = Abuf + mo, *pm = phimap + mo, *pmT = phimapT + mo;
    const float *lv = leaves + (size_t)cp * 2 * P.Np, *jw = jaws + 4 * cp;
    const int bw = d.a1 - d.a0 + 1, bh = d.b1 - d.b0 + 1, npx = bw * bh;
    const int pw = d.pa1 - d.pa0 + 1, ph = d.pb1 - d.pb0 + 1, npp = pw * ph;
    const float x1 = jw[0], x2 = jw[1], y1 = jw[2], y2 = jw[3];
    const bool rotated = d.sc != 0.f || d.cc != 1.f;
    // The intermediate maps (Phi0, the blur temporaries, the map itself) live in shared memory when the support bbox fits: every
    // pass is then a chain of shared-memory round trips instead of L2 ones.  Larger fields work in the global scratch planes.
    __shared__ float tile[3][FLU_TILE];
    const bool in_smem = npx <= FLU_TILE && npp <= FLU_TILE;
    const MapView vP0 = in_smem ? MapView{ tile[0], bw, d.a0, d.b0 } : MapView{ P0 + mo, P.Nuf, 0, 0 };
    const MapView vT = in_smem ? MapView{ tile[1], bw, d.a0, d.b0 } : MapView{ T1 + mo, P.Nuf, 0, 0 };
    const MapView vM = in_smem ? MapView{ tile[2], bw, d.a0, d.b0 } : MapView{ pm, P.Nuf, 0, 0 };

    // leaf pairs that can overlap each pixel row of the jaw opening (the bounds are ascending): once per row
    __shared__ short leaf_lo[FLU_MAX_ROWS], leaf_hi[FLU_MAX_ROWS];
    const bool ranged = d.jb1 - d.jb0 < FLU_MAX_ROWS;
    if (ranged) {
        for (int r = tid; r <= d.jb1 - d.jb0; r += FLU_THREADS) {
            const float vf = flu_v(P, d.jb0 + r), vlo = vf - 0.5f * P.Dv, vhi = vf + 0.5f * P.Dv;
            int lo = 0, hi = P.Np - 1;
            while (lo < P.Np && T.leaf_bounds[lo + 1] <= vlo) ++lo;
            while (hi >= 0 && T.leaf_bounds[hi] >= vhi) --hi;
            leaf_lo[r] = (short)lo; leaf_hi[r] = (short)hi;
        }
    }
    __syncthreads();
    // O1, O2: A, J, Phi0
    for (int p = tid; p < npx; p += FLU_THREADS) {
        const int a = d.a0 + p % bw, b = d.b0 + p / bw;
        float A = 0.f, J = 0.f;
        if (a >= d.ja0 && a <= d.ja1 && b >= d.jb0 && b <= d.jb1) {
            const float uf = flu_u(P, a), vf = flu_v(P, b);
            const int i0 = ranged ? leaf_lo[b - d.jb0] : 0, i1 = ranged ? leaf_hi[b - d.jb0] : P.Np - 1;
            for (int i = i0; i <= i1; ++i) {
                const float ovv = ov(vf, P.Dv, T.leaf_bounds[i], T.leaf_bounds[i + 1]);
                if (ovv != 0.f) A += ovv * ov(uf, P.Du, lv[i], lv[P.Np + i]);
            }
            J = ov(uf, P.Du, x1, x2) * ov(vf, P.Dv, y1, y2);
        }
        Am[b * P.Nuf + a] = A;                               // read again by k_fluence_adjoint
        vP0.at(a, b) = J * (P.tau + (1.f - P.tau) * A);
    }
    __syncthreads();
    // O3: penumbra, u with the MLC width then v with the jaw width
    for (int p = tid; p < npx; p += FLU_THREADS) {
        const int a = d.a0 + p % bw, b = d.b0 + p / bw;
        vT.at(a, b) = view_blur(vP0, d, a, b, 0, T.Tu, T.gu);
    }
    __syncthreads();
    for (int p = tid; p < npx; p += FLU_THREADS) {
        const int a = d.a0 + p % bw, b = d.b0 + p / bw;
        vM.at(a, b) = view_blur(vT, d, a, b, 1, T.Tv, T.gv);
    }
    // O4: head scatter
    for (int q = 0; q < T.n_hs; ++q) {
        __syncthreads();
        for (int p = tid; p < npx; p += FLU_THREADS) {
            const int a = d.a0 + p % bw, b = d.b0 + p / bw;
            vT.at(a, b) = view_blur(vP0, d, a, b, 1, T.hs_Tv[q], T.hs_gv[q]);
        }
        __syncthreads();
        for (int p = tid; p < npx; p += FLU_THREADS) {
            const int a = d.a0 + p % bw, b = d.b0 + p / bw;
            vM.at(a, b) += T.hs_amp[q] * view_blur(vT, d, a, b, 0, T.hs_Tu[q], T.hs_gu[q]);
        }
    }
    __syncthreads();
    // O5: off-axis
    for (int p = tid; p < npx; p += FLU_THREADS) {
        const int a = d.a0 + p % bw, b = d.b0 + p / bw;
        const float uf = flu_u(P, a), vf = flu_v(P, b);
        vM.at(a, b) *= oar_factor(T, sqrtf(uf * uf + vf * vf));
    }
    __syncthreads();
    // collimator rotation (G25): the map is resampled (bilinear_0) on its own grid at R(-phi_c) of
    // each pixel centre; from here on the map lives in the projection frame (bbox pa0..pb1)
    MapView vF = vM;                                         // the final map
    if (rotated) {
        const MapView vR = in_smem ? MapView{ tile[1], pw, d.pa0, d.pb0 } : MapView{ T1 + mo, P.Nuf, 0, 0 };
        for (int p = tid; p < npp; p += FLU_THREADS) {
            const int a = d.pa0 + p % pw, b = d.pb0 + p / pw;
            const float u = flu_u(P, a), v = flu_v(P, b);
            const float fa = (d.cc * u + d.sc * v) / P.Du + P.cuf, fb = (-d.sc * u + d.cc * v) / P.Dv + P.cvf;
            const float fla = floorf(fa), flb = floorf(fb);
            const int ia = (int)fla, ib = (int)flb;
            const float ta = fa - fla, tb = fb - flb;
            vR.at(a, b) = (1.f - tb) * ((1.f - ta) * view_at(vM, d.a0, d.a1, d.b0, d.b1, ia, ib) + ta * view_at(vM, d.a0, d.a1, d.b0, d.b1, ia + 1, ib)) +
                          tb * ((1.f - ta) * view_at(vM, d.a0, d.a1, d.b0, d.b1, ia, ib + 1) + ta * view_at(vM, d.a0, d.a1, d.b0, d.b1, ia + 1, ib + 1));
        }
        __syncthreads();
        vF = vR;
        if (!in_smem) {     // the global plane of the map held the collimator-frame values: clear them, the projection-frame box follows
            for (int p = tid; p < npx; p += FLU_THREADS) pm[(d.b0 + p / bw) * P.Nuf + d.a0 + p % bw] = 0.f;
            __syncthreads();
        }
    }
    // the map [b][a] (k_fluence_adjoint, stage tap) and the same with v fastest (k_project stages that one)
    if (in_smem || rotated) {
        for (int p = tid; p < npp; p += FLU_THREADS) {
            const int a = d.pa0 + p % pw, b = d.pb0 + p / pw;
            pm[b * P.Nuf + a] = vF.at(a, b);
        }
    }
    for (int p = tid; p < npp; p += FLU_THREADS) {
        const int a = d.pa0 + p / ph, b = d.pb0 + p % ph;
        pmT[a * P.Nvf + b] = vF.at(a, b);
    }
}

// Exclusive prefix of the conv work items over the control points [cp0, cp0+n) and the totals.
// One block of 256 threads: warp-shuffle scan per 256-entry chunk with a running carry.
__global__ void __launch_bounds__(256) k_scan_items(const CpDesc *desc, int cp0, int n, int adjoint, int nuf, int nvf, int *tile_base, WorkCounters *wc)
{
    __shared__ int wsum[8];
    __shared__ unsigned long long tot[6];
    __shared__ int carry_s;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid < 6) tot[tid] = 0ull;
    if (tid == 0) carry_s = 0;
    __syncthreads();
    unsigned long long acc[6] = { 0ull, 0ull, 0ull, 0ull, 0ull, 0ull };
    for (int c0 = 0; c0 < n; c0 += 256) {
        const int c = c0 + tid;
        int v = 0;
        if (c < n) {
            const CpDesc &d = desc[cp0 + c];
            v = adjoint ? d.n_items_adj : d.n_items;
            acc[0] += d.support_vox; acc[1] += d.footprint_vox; acc[2] += d.region_vox; acc[3] += d.macs_fwd; acc[4] += d.macs_adj;
            if (d.a0 <= d.a1)       // rays of the divergent-depth mode: the support bbox grown by one pixel, clipped to the map
                acc[5] += (unsigned long long)(min(nuf - 1, d.pa1 + 1) - max(0, d.pa0 - 1) + 1) * (min(nvf - 1, d.pb1 + 1) - max(0, d.pb0 - 1) + 1);
        }
        int incl = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        if (lane == 31) wsum[warp] = incl;
        __syncthreads();
        int woff = 0;
        for (int w = 0; w < warp; ++w) woff += wsum[w];
        const int carry = carry_s;
        if (c < n) tile_base[c] = carry + woff + incl - v;
        __syncthreads();
        if (tid == 255) carry_s = carry + woff + incl;
        __syncthreads();
    }
#pragma unroll
    for (int q = 0; q < 6; ++q) {
        unsigned long long v = acc[q];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) atomicAdd(&tot[q], v);
    }
    __syncthreads();
    if (tid == 0) {
        tile_base[n] = carry_s;
        tile_base[n + 1] = 0;           // unit counter of the conv launch that follows
        if (cp0 == 0) { wc->items = 0; wc->support_vox = 0; wc->footprint_vox = 0; wc->region_vox = 0; wc->macs_fwd = 0; wc->macs_adj = 0; wc->fan_rays = 0; }
        wc->items += carry_s; wc->support_vox += tot[0]; wc->footprint_vox += tot[1];
        wc->region_vox += tot[2]; wc->macs_fwd += tot[3]; wc->macs_adj += tot[4]; wc->fan_rays += tot[5];
    }
}

// S10.  d_mu = cal <Phimap, gPhimap>; then cal*MU*gPhimap back through OAR, the (self-adjoint,
// zero-padded) Gaussians, the product Phi0 = J (tau + (1-tau) A) and Eq. 4's subgradients.
// One block per control point; leaf gradients need no reduction (one thread per leaf edge),
// jaw and MU gradients use warp-shuffle + shared-memory block reductions (no global atomics).
__global__ void __launch_bounds__(FLU_THREADS, 2)
k_fluence_adjoint(Params P, FluTables T, int n_cp, const float *__restrict__ leaves, const float *__restrict__ jaws,
                  const CpDesc *__restrict__ desc, const float *__restrict__ phimap, const float *__restrict__ Abuf,
                  const float *__restrict__ gphimap, float *T1, float *T2, float *T3,
                  float *d_leaves, float *d_jaws, float *d_mu)
{
    const int cp = blockIdx.x, tid = threadIdx.x;
    if (cp >= n_cp) return;
    __shared__ CpDesc d;
    __shared__ float red[5][FLU_THREADS / 32];
    if (tid == 0) d = desc[cp];
    __syncthreads();
    float *dl = d_leaves + (size_t)cp * 2 * P.Np;
    if (d.a0 > d.a1) {      // closed jaws: nothing reaches the patient
        for (int e = tid; e < 2 * P.Np; e += FLU_THREADS) dl[e] = 0.f;
        if (tid < 4) d_jaws[4 * cp + tid] = 0.f;
        if (tid == 0) d_mu[cp] = 0.f;
        return;
    }
    const size_t mo = (size_t)cp * P.Nuf * P.Nvf;
    const float *pm = phimap + mo, *Am = Abuf + mo, *gp = gphimap + mo;
    float *g2 = T1 + mo, *t = T2 + mo, *gP0 = T3 + mo;
    const float *lv = leaves + (size_t)cp * 2 * P.Np, *jw = jaws + 4 * cp;
    const int bw = d.a1 - d.a0 + 1, bh = d.b1 - d.b0 + 1, npx = bw * bh;
    const float x1 = jw[0], x2 = jw[1], y1 = jw[2], y2 = jw[3];
    float acc[5] = { 0.f, 0.f, 0.f, 0.f, 0.f };     // d_x1, d_x2, d_y1, d_y2, <Phimap, gPhimap>

    const bool rotated = d.sc != 0.f || d.cc != 1.f;
    if (rotated) {      // <Phimap, gPhimap> over the projection-frame bbox (both live in the projection frame)
        const int pw = d.pa1 - d.pa0 + 1, npp = pw * (d.pb1 - d.pb0 + 1);
        for (int p = tid; p < npp; p += FLU_THREADS) {
            const int a = d.pa0 + p % pw, b = d.pb0 + p / pw;
            acc[4] += pm[b * P.Nuf + a] * gp[b * P.Nuf + a];
        }
    }
    // half-extent, in pixels of the projection frame, of a collimator-frame pixel's hat after the rotation
    const float hra = (fabsf(d.cc) * P.Du + fabsf(d.sc) * P.Dv) / P.Du, hrb = (fabsf(d.sc) * P.Du + fabsf(d.cc) * P.Dv) / P.Dv;
    for (int p = tid; p < npx; p += FLU_THREADS) {          // (rotation transposed,) O5 transposed, scaled by cal*MU
        const int a = d.a0 + p % bw, b = d.b0 + p / bw;
        const float uf = flu_u(P, a), vf = flu_v(P, b);
        float gv;
        if (!rotated) {
            gv = gp[b * P.Nuf + a];
            acc[4] += pm[b * P.Nuf + a] * gv;
        } else {
            // gather form of the transpose: the projection-frame pixels (a', b') whose sample point R(-phi_c)(uf_a', vf_b')
            // lies within one pixel of (a, b) sit around R(phi_c)(uf_a, vf_b)
            const float far = (d.cc * uf - d.sc * vf) / P.Du + P.cuf, fbr = (d.sc * uf + d.cc * vf) / P.Dv + P.cvf;
            const int a_lo = max(d.pa0, (int)ceilf(far - hra)), a_hi = min(d.pa1, (int)floorf(far + hra));
            const int b_lo = max(d.pb0, (int)ceilf(fbr - hrb)), b_hi = min(d.pb1, (int)floorf(fbr + hrb));
            gv = 0.f;
            for (int bb = b_lo; bb <= b_hi; ++bb)
                for (int aa = a_lo; aa <= a_hi; ++aa) {
                    const float u = flu_u(P, aa), v = flu_v(P, bb);
                    const float wa = 1.f - fabsf((d.cc * u + d.sc * v) / P.Du + P.cuf - (float)a);
                    const float wb = 1.f - fabsf((-d.sc * u + d.cc * v) / P.Dv + P.cvf - (float)b);
                    if (wa > 0.f && wb > 0.f) gv = fmaf(wa * wb, gp[bb * P.Nuf + aa], gv);
                }
        }
        g2[b * P.Nuf + a] = d.scale * gv * oar_factor(T, sqrtf(uf * uf + vf * vf));
    }
    __syncthreads();
    for (int p = tid; p < npx; p += FLU_THREADS) {          // O3 transposed: v (jaw) ...
        const int a = d.a0 + p % bw, b = d.b0 + p / bw;
        t[b * P.Nuf + a] = blur_at(g2, P, d, a, b, 1, T.Tv, T.gv);
    }
    __syncthreads();
    for (int p = tid; p < npx; p += FLU_THREADS) {          // ... then u (MLC)
        const int a = d.a0 + p % bw, b = d.b0 + p / bw;
        gP0[b * P.Nuf + a] = blur_at(t, P, d, a, b, 0, T.Tu, T.gu);
    }
    for (int q = 0; q < T.n_hs; ++q) {                      // O4 transposed
        __syncthreads();
        for (int p = tid; p < npx; p += FLU_THREADS) {
            const int a = d.a0 + p % bw, b = d.b0 + p / bw;
            t[b * P.Nuf + a] = blur_at(g2, P, d, a, b, 0, T.hs_Tu[q], T.hs_gu[q]);
        }
        __syncthreads();
        for (int p = tid; p < npx; p += FLU_THREADS) {
            const int a = d.a0 + p % bw, b = d.b0 + p / bw;
            gP0[b * P.Nuf + a] += T.hs_amp[q] * blur_at(t, P, d, a, b, 1, T.hs_Tv[q], T.hs_gv[q]);
        }
    }
    __syncthreads();
    // O2: jaws (product rule; d ov is non-zero on one pixel column / row only)
    const int jw_w = d.ja1 - d.ja0 + 1, jw_n = jw_w * (d.jb1 - d.jb0 + 1);
    for (int p = tid; p < jw_n; p += FLU_THREADS) {
        const int a = d.ja0 + p % jw_w, b = d.jb0 + p / jw_w;
        const float uf = flu_u(P, a), vf = flu_v(P, b);
        const float ju = ov(uf, P.Du, x1, x2), jv = ov(vf, P.Dv, y1, y2);
        const float gJ = gP0[b * P.Nuf + a] * (P.tau + (1.f - P.tau) * Am[b * P.Nuf + a]);
        acc[0] += gJ * dov_dlo(uf, P.Du, x1, x2) * jv;
        acc[1] += gJ * dov_dhi(uf, P.Du, x1, x2) * jv;
        acc[2] += gJ * ju * dov_dlo(vf, P.Dv, y1, y2);
        acc[3] += gJ * ju * dov_dhi(vf, P.Dv, y1, y2);
    }
    // O1: leaves — one thread per leaf edge, a handful of pixel rows each
    const float eu = -0.5f * P.Nuf * P.Du, ev = -0.5f * P.Nvf * P.Dv;
    for (int e = tid; e < 2 * P.Np; e += FLU_THREADS) {
        const int bank = e / P.Np, i = e % P.Np;
        const float lo = lv[i], hi = lv[P.Np + i];
        // pixel that holds the edge, clamped in float first: positions are unvalidated (inf, huge values)
        const float fc = fminf(fmaxf(((bank == 0 ? lo : hi) - eu) / P.Du, -2.f), (float)P.Nuf + 2.f);
        const int ac = bank == 0 ? (int)ceilf(fc) - 1 : (int)floorf(fc);
        float s = 0.f;
        for (int a = max(ac - 1, d.ja0); a <= min(ac + 1, d.ja1); ++a) {      // the index arithmetic may be off by one at a pixel edge
            const float uf = flu_u(P, a);
            const float dv_ = bank == 0 ? dov_dlo(uf, P.Du, lo, hi) : dov_dhi(uf, P.Du, lo, hi);
            if (dv_ == 0.f) continue;
            const float ju = ov(uf, P.Du, x1, x2);
            const int blo = max(d.jb0, (int)floorf((T.leaf_bounds[i] - ev) / P.Dv) - 1);
            const int bhi = min(d.jb1, (int)floorf((T.leaf_bounds[i + 1] - ev) / P.Dv) + 1);
            for (int b = blo; b <= bhi; ++b) {
                const float vf = flu_v(P, b);
                const float ovv = ov(vf, P.Dv, T.leaf_bounds[i], T.leaf_bounds[i + 1]);
                const float gA = gP0[b * P.Nuf + a] * ju * ov(vf, P.Dv, y1, y2) * (1.f - P.tau);
                s += gA * ovv * dv_;
            }
        }
        dl[e] = s;
    }
    // block reduction of the five scalars
#pragma unroll
    for (int q = 0; q < 5; ++q) {
        const float v = warp_sum(acc[q]);
        if ((tid & 31) == 0) red[q][tid >> 5] = v;
    }
    __syncthreads();
    if (tid < 5) {
        float s = 0.f;
        for (int w = 0; w < FLU_THREADS / 32; ++w) s += red[tid][w];
        if (tid < 4) d_jaws[4 * cp + tid] = s;
        else d_mu[cp] = P.cal * s;
    }
}

}  // namespace pdrt
