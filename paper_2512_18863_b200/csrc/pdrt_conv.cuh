// pdrt_conv.cuh — S3 (divergent projection), S4+S5 (depth-indexed kernel lookup + lateral convolution),
// S7 (transpose of the beam -> patient resampling) and S8 (convolution adjoint).
//
// Forward (PAPER.md:123-133 Eq. 5-6, :145-149, :151-158 Eq. 8), per control point b and slice k:
//   Phivol(i,j) = mag^2 * bilinear_0(Phimap_b; mag u_i/Du + cuf, mag v_j/Dv + cvf),  mag = SID/(SID+w_k)   k_project
//   W_k         = lerp of the pre-integrated table W_tab at t = z_rad(b,k)/dz                               k_conv
//   D_b(i,j,k)  = sum_{dj,di} W_k[dj][di] * Phivol(i+di-c, j+dj-c)                                         k_conv
// Adjoint: G_b = R_b^T g (k_resample_adjoint), H_b = conv of G_b with the flipped kernel, outputs on S_k only.
//
// Phivol and G_b are written once, over S_k resp. F_k only, in the compact v-fastest block layout
// (pdrt_dev.cuh); that lets the convolution stage its input tiles with cp.async (zero-filled outside the
// source box).
//
// The convolution is bound by the FP32 FMA pipe (k^2 multiply-adds per 4-byte output), so the
// kernel is organised around FMA-pipe cycles: each thread owns an RF x RS = 8(v) x 2(u) register tile, slides a
// (K+7)-wide register window along v (LDS.128), takes weight PAIRS as warp-broadcast LDS.128 and issues packed
// FFMA2 (fma.rn.f32x2: both output rows of the thread-tile in one instruction).
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

// 4-byte asynchronous global -> shared copy; `ok == false` writes a zero instead (no global read).
__device__ __forceinline__ void cp_async_f32(float *dst_smem, const float *src, bool ok)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst_smem);
    const int n = ok ? 4 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;\n" ::"r"(d), "l"(src), "r"(n) : "memory");
}
// the same with shared-window addresses and an explicit source size (bytes actually read; the rest is zero-filled)
__device__ __forceinline__ void cp_async_4(unsigned dst, const float *src, int n)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;\n" ::"r"(dst), "l"(src), "r"(n) : "memory");
}
__device__ __forceinline__ void cp_async_8(unsigned dst, const float *src, int n)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(dst), "l"(src), "r"(n) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }

constexpr int PROJECT_THREADS = 128;
constexpr int PROJECT_MAP_FLOATS = 4096;          // support bbox of the fluence map staged in shared memory when it fits (16 KB)

// S3.  Phivol over S_k (Eq. 5-6) into the compact block of the control point.  The bilinear sample is separable:
//   Phivol(i,j) = (1-ta) T[a][j] + ta T[a+1][j],   T[a][j] = mag^2 ((1-tb) Phimap[a][b] + tb Phimap[a][b+1]),
// with (a, ta) a function of the row i and (b, tb) of the column j.  A THREAD owns one 16-byte quad of four consecutive v
// (the contiguous axis) of one slice and walks down the rows i of S_k: the column terms of its four voxels are worked out
// once, the pixel row a(i) never decreases along the walk, so the thread keeps T[a] and T[a+1] of its quad in registers and
// evaluates each pixel row once (8 map reads), and every voxel row costs 8 multiply-adds and one aligned float4 store.
// A block works on PROJECT_THREADS / qw slices at a time (qw = quads per row of the widest slice).  The support bbox of
// the map (a few KB) is staged in shared memory once per block with all its loads in flight together: the walk is a
// chain of dependent reads, which from shared memory cost 30 cycles each instead of an L2 round trip.  Columns [S.v0 & ~3, S.v1 | 3] are written (the conv stages its tiles in aligned pairs; the extra
// columns are structural zeros and lie inside the region because rj0 % 8 == 0 and pv % 8 == 0).  Grid: (X, n_cp).
__global__ void __launch_bounds__(PROJECT_THREADS)
k_project(Params P, const CpDesc *__restrict__ desc, const SliceBox16 *__restrict__ sbox, int cp0, int n_cp,
          const float *__restrict__ phimapT, float *__restrict__ vol)
{
    const int slot = blockIdx.y;
    if (slot >= n_cp) return;
    const int cp = cp0 + slot;
    const CpDesc d = desc[cp];
    if (d.a0 > d.a1) return;
    const float *pm = phimapT + (size_t)cp * P.Nuf * P.Nvf;
    float *vc = vol + (size_t)slot * (size_t)P.stride_cp;
    __shared__ float map_s[PROJECT_MAP_FLOATS];              // [a - a0][b - b0], b fastest
    const int bw = d.pa1 - d.pa0 + 1, bh = d.pb1 - d.pb0 + 1;
    const bool staged = bw * bh <= PROJECT_MAP_FLOATS;
    if (staged) {
        for (int a = threadIdx.x >> 5; a < bw; a += PROJECT_THREADS / 32)
            for (int b = threadIdx.x & 31; b < bh; b += 32) map_s[a * bh + b] = __ldg(pm + (d.pa0 + a) * P.Nvf + d.pb0 + b);
    }
    __syncthreads();
    // quads per row of the widest slice: S_k grows with the distance from the source, and its first column may round down
    const SliceBox16 Sl = load_box(sbox, (size_t)cp * P.Nw + P.Nw - 1), Sf = load_box(sbox, (size_t)cp * P.Nw);
    const int wide = max(Sl.u0 <= Sl.u1 ? Sl.v1 - Sl.v0 + 1 : 0, Sf.u0 <= Sf.u1 ? Sf.v1 - Sf.v0 + 1 : 0);
    const int qw = min(PROJECT_THREADS, (wide + 3) / 4 + 1);
    const int spb = PROJECT_THREADS / qw;                       // slices per block iteration
    const int ks = threadIdx.x / qw, jq = threadIdx.x - ks * qw;
    if (ks >= spb) return;
    for (int k = blockIdx.x * spb + ks; k < P.Nw; k += gridDim.x * spb) {
        const SliceBox16 S = load_box(sbox, (size_t)cp * P.Nw + k);
        if (S.u0 > S.u1) continue;
        const float mag = P.sid / (P.sid + P.wmin + k * P.dw), m2 = mag * mag;
        const float su = mag * P.du / P.Du, sv = mag / P.Dv;
        const int j0 = S.v0 & ~3, nq = (((int)S.v1 | 3) - j0 + 1) >> 2;
        for (int q = jq; q < nq; q += qw) {                    // one pass (a second one only if a slice is wider than the bound)
            // column terms of this thread's four voxels: m2-scaled weights of pixel rows b and b+1; invalid rows get weight 0
            // and are folded onto a valid one, so that every address is readable
            const int jb = j0 + 4 * q;
            float wb0[4], wb1[4];
            int ib0[4], ib1[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int j = jb + e;
                const float fb = (P.v0 + j * P.dv) * sv + P.cvf;
                const float flb = floorf(fb);
                const int b = (int)flb;
                const float tb = fb - flb;
                const bool jgrid = j < P.Nv;
                const bool v0 = jgrid && b >= d.pb0 && b <= d.pb1, v1 = jgrid && b + 1 >= d.pb0 && b + 1 <= d.pb1;
                wb0[e] = v0 ? m2 * (1.f - tb) : 0.f; wb1[e] = v1 ? m2 * tb : 0.f;
                ib0[e] = v0 ? b : (v1 ? b + 1 : d.pb0); ib1[e] = v1 ? b + 1 : ib0[e];
            }
            auto row_T = [&](int a, float (&T)[4]) {            // T[a][quad]; zero outside the support bbox
                if (a >= d.pa0 && a <= d.pa1) {
                    if (staged) {
                        const float *pc = map_s + (a - d.pa0) * bh - d.pb0;
#pragma unroll
                        for (int e = 0; e < 4; ++e) T[e] = wb0[e] * pc[ib0[e]] + wb1[e] * pc[ib1[e]];
                    } else {
                        const float *pc = pm + a * P.Nvf;
#pragma unroll
                        for (int e = 0; e < 4; ++e) T[e] = wb0[e] * __ldg(pc + ib0[e]) + wb1[e] * __ldg(pc + ib1[e]);
                    }
                } else {
#pragma unroll
                    for (int e = 0; e < 4; ++e) T[e] = 0.f;
                }
            };
            int a_cur = (int)floorf((S.u0 - P.cu) * su + P.cuf);
            float T0[4], T1[4];
            row_T(a_cur, T0);
            row_T(a_cur + 1, T1);
            float *op = vc + ((size_t)k * d.pu + (S.u0 - d.ri0)) * d.pv + (jb - d.rj0);
            const float fa0 = (S.u0 - P.cu) * su + P.cuf;
            for (int i = S.u0; i <= S.u1; ++i, op += d.pv) {
                const float fa = fmaf((float)(i - S.u0), su, fa0);
                const float fla = floorf(fa);
                const int a = (int)fla;
                const float ta = fa - fla;
                while (a_cur < a) {                            // a(i) never decreases along the walk
#pragma unroll
                    for (int e = 0; e < 4; ++e) T0[e] = T1[e];
                    ++a_cur;
                    row_T(a_cur + 1, T1);
                }
                *reinterpret_cast<float4 *>(op) = make_float4(T0[0] + ta * (T1[0] - T0[0]), T0[1] + ta * (T1[1] - T0[1]),
                                                               T0[2] + ta * (T1[2] - T0[2]), T0[3] + ta * (T1[3] - T0[3]));
            }
        }
    }
}

constexpr int RA_THREADS = 256, RA_MAXC = 9, RA_PADC = 12;
struct __align__(16) RaRow {        // one beam row (k, i) of G_b: its patient-column candidates, compacted
    int off[RA_PADC];               // offsets of gT[y][x][0]; entries past n repeat entry 0 ...
    float w[RA_PADC];               // ... with weight 0, so that the stream loop needs no predicates
    int n;                          // candidates with a non-zero weight; -1: nothing to write; -2: stencil wider than 3 x 3
    int out;                        // offset of G_b(k, i, v = 0) in the control point's compact block
    int j0, nq;                     // first column (multiple of 4) and number of quads to write
    int xa, xb, ya, yb;             // candidate box of the general path
    float eu0, ew0;
    int pad_[2];                    // 144 bytes: an odd number of 16-byte chunks, so that the set-up's stores (one row per thread) spread
                                    // over the banks
};
static_assert(sizeof(RaRow) == 144, "row records are 9 chunks of 16 bytes");

// one quad of each of TWO beam rows from NC candidates each (the first NC entries of the rows' lists), no predicates: the
// 2 NC loads are all in flight before the first use.  A row with nothing to write has nq = 0.
template <int NC>
__device__ __forceinline__ void ra_stream2(const RaRow &Ra, const RaRow &Rb, const float *__restrict__ gT, float *__restrict__ Gc, int lane16)
{
    const int nqa = Ra.n >= 0 ? Ra.nq : 0, nqb = Rb.n >= 0 ? Rb.nq : 0;
    float *oa = Gc + Ra.out, *ob = Gc + Rb.out;
    for (int q = lane16; q < max(nqa, nqb); q += 16) {
        const int ja = Ra.j0 + 4 * min(q, max(nqa - 1, 0)), jb = Rb.j0 + 4 * min(q, max(nqb - 1, 0));
        int offa[NC], offb[NC];
        float wa[NC], wb[NC];
#pragma unroll
        for (int c4 = 0; c4 < NC; c4 += 4) {                  // 16-byte broadcast reads of the lists
            const int4 o = *reinterpret_cast<const int4 *>(&Ra.off[c4]), p = *reinterpret_cast<const int4 *>(&Rb.off[c4]);
            const float4 f = *reinterpret_cast<const float4 *>(&Ra.w[c4]), g = *reinterpret_cast<const float4 *>(&Rb.w[c4]);
            offa[c4] = o.x; wa[c4] = f.x; offb[c4] = p.x; wb[c4] = g.x;
            if (c4 + 1 < NC) { offa[c4 + 1] = o.y; wa[c4 + 1] = f.y; offb[c4 + 1] = p.y; wb[c4 + 1] = g.y; }
            if (c4 + 2 < NC) { offa[c4 + 2] = o.z; wa[c4 + 2] = f.z; offb[c4 + 2] = p.z; wb[c4 + 2] = g.z; }
            if (c4 + 3 < NC) { offa[c4 + 3] = o.w; wa[c4 + 3] = f.w; offb[c4 + 3] = p.w; wb[c4 + 3] = g.w; }
        }
        float4 va[NC], vb[NC];
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            va[c] = __ldg(reinterpret_cast<const float4 *>(gT + (offa[c] + ja)));
            vb[c] = __ldg(reinterpret_cast<const float4 *>(gT + (offb[c] + jb)));
        }
        float4 sa = make_float4(0.f, 0.f, 0.f, 0.f), sb = sa;
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            sa.x = fmaf(wa[c], va[c].x, sa.x); sa.y = fmaf(wa[c], va[c].y, sa.y); sa.z = fmaf(wa[c], va[c].z, sa.z); sa.w = fmaf(wa[c], va[c].w, sa.w);
            sb.x = fmaf(wb[c], vb[c].x, sb.x); sb.y = fmaf(wb[c], vb[c].y, sb.y); sb.z = fmaf(wb[c], vb[c].z, sb.z); sb.w = fmaf(wb[c], vb[c].w, sb.w);
        }
        if (q < nqa) *reinterpret_cast<float4 *>(oa + ja) = sa;
        if (q < nqb) *reinterpret_cast<float4 *>(ob + jb) = sb;
    }
}

// S7.  G_b = R_b^T g over F_k in gather form: G_b(i,j,k) = sum over the patient voxels (x,y) of slice z = j whose
// bilinear stencil (as evaluated by k_gather_dose) reaches beam voxel (i,k), weight (1-|du|)(1-|dw|), times g.
// The gantry rotates about patient z = beam v (G1), so the weights do not depend on v.  A block takes 256
// beam rows (k, i) of the control point's region at a time.  Phase A: one THREAD per row works out the (at most 3 x 3)
// candidate columns and keeps those with a non-zero weight (4 on average) in shared memory.  Phase B: one HALF-WARP per
// row streams 16-byte vectors along v: coalesced reads of gT[y][x][v] (dL/dDose with z fastest, row pitch padded to a
// multiple of 4, L2-resident) and one aligned float4 store per lane; the loop is specialised on the number of candidates
// (4, 6 or 9: the list is padded with zero weights) so that it carries no predicates.
// Grid: (X, n_cp), blocks stride over the row chunks.
__global__ void __launch_bounds__(RA_THREADS, 4)
k_resample_adjoint(Params P, const CpDesc *__restrict__ desc, const SliceBox16 *__restrict__ sbox, int cp0, int n_cp, int C,
                   int nzp, const float *__restrict__ gT, float *__restrict__ G)
{
    __shared__ RaRow rows[RA_THREADS];
    const int slot = blockIdx.y;
    if (slot >= n_cp) return;
    const int cp = cp0 + slot;
    const CpDesc d = desc[cp];
    if (d.a0 > d.a1) return;
    const int tid = threadIdx.x, lane16 = tid & 15, half = tid >> 4;
    // half-extent, in patient indices, of the rotated unit hat of one beam voxel; beam-index increments per patient step
    const float hx = (fabsf(d.cg) * P.du + fabsf(d.sg) * P.dw) / P.sx, hy = (fabsf(d.sg) * P.du + fabsf(d.cg) * P.dw) / P.sy;
    const float fu_x = d.cg * P.sx / P.du, fu_y = d.sg * P.sy / P.du, fw_x = -d.sg * P.sx / P.dw, fw_y = d.cg * P.sy / P.dw;
    // affine maps: patient index of beam voxel (i,k), beam index of patient voxel (x,y)
    const float fx_i = P.du * d.cg / P.sx, fy_i = P.du * d.sg / P.sy;
    const float fx_0 = (P.isox - P.cu * P.du * d.cg - P.ox) / P.sx, fy_0 = (P.isoy - P.cu * P.du * d.sg - P.oy) / P.sy;
    const float fx_w = -d.sg / P.sx, fy_w = d.cg / P.sy;
    const float fu_0 = (d.cg * (P.ox - P.isox) + d.sg * (P.oy - P.isoy)) / P.du + P.cu;
    const float fw_0 = (-d.sg * (P.ox - P.isox) + d.cg * (P.oy - P.isoy) - P.wmin) / P.dw;
    float *Gc = G + (size_t)slot * (size_t)P.stride_cp;
    const int n_rows = P.Nw * d.pu;
    for (int r0 = blockIdx.x * RA_THREADS; r0 < n_rows; r0 += gridDim.x * RA_THREADS) {
        __syncthreads();                                     // the previous chunk has been streamed
        {   // phase A
            RaRow &R = rows[tid];
            const int r = r0 + tid;
            int n = -1;
            R.out = 0; R.j0 = 0; R.nq = 0;
            if (r < n_rows) {
                const int k = r / d.pu, i = d.ri0 + (r - k * d.pu);
                const SliceBox16 S = load_box(sbox, (size_t)cp * P.Nw + k);
                const int fu0 = max(0, S.u0 - C), fu1 = min(P.Nu - 1, S.u1 + C), fv0 = max(0, S.v0 - C), fv1 = min(P.Nv - 1, S.v1 + C);
                if (S.u0 <= S.u1 && i >= fu0 && i <= fu1) {
                    R.out = (k * d.pu + (i - d.ri0)) * d.pv - d.rj0;
                    R.j0 = fv0 & ~3; R.nq = ((fv1 | 3) - R.j0 + 1) >> 2;
                    const float w = P.wmin + k * P.dw;
                    const float fx = fx_0 + w * fx_w + i * fx_i, fy = fy_0 + w * fy_w + i * fy_i;
                    const int xa = max(0, (int)ceilf(fx - hx)), xb = min(P.nx - 1, (int)floorf(fx + hx));
                    const int ya = max(0, (int)ceilf(fy - hy)), yb = min(P.ny - 1, (int)floorf(fy + hy));
                    const float eu0 = fu_0 + xa * fu_x + ya * fu_y - (float)i;
                    const float ew0 = fw_0 + xa * fw_x + ya * fw_y - (float)k;
                    n = 0;
                    if (xb - xa <= 2 && yb - ya <= 2) {
                        for (int cy = 0; cy <= yb - ya; ++cy)
                            for (int cx = 0; cx <= xb - xa; ++cx) {
                                const float wu = 1.f - fabsf(eu0 + cy * fu_y + cx * fu_x), ww = 1.f - fabsf(ew0 + cy * fw_y + cx * fw_x);
                                if (wu > 0.f && ww > 0.f) { R.off[n] = ((ya + cy) * P.nx + xa + cx) * nzp; R.w[n] = wu * ww; ++n; }
                            }
                    } else {
                        n = -2;
                        R.xa = xa; R.xb = xb; R.ya = ya; R.yb = yb; R.eu0 = eu0; R.ew0 = ew0;
                    }
                }
            }
            {   // entries past n repeat entry 0 with weight 0 (every address readable, no predicates in the stream loop)
                const int o0 = n > 0 ? R.off[0] : 0;
                for (int c = max(n, 0); c < RA_MAXC; ++c) { R.off[c] = o0; R.w[c] = 0.f; }
            }
            R.n = n;
        }
        __syncthreads();
        // phase B: half-warp `half` streams the row pairs (half, half + 16), (half + 32, half + 48), ...
        for (int rr = half; rr < RA_THREADS; rr += RA_THREADS / 8) {
            const RaRow &Ra = rows[rr], &Rb = rows[rr + RA_THREADS / 16];
            const int na = Ra.n, nb = Rb.n;
            if (na == -1 && nb == -1) continue;
            if (na != -2 && nb != -2) {
                const int n = max(na, nb);
                if (n <= 4) ra_stream2<4>(Ra, Rb, gT, Gc, lane16);
                else if (n <= 6) ra_stream2<6>(Ra, Rb, gT, Gc, lane16);
                else ra_stream2<RA_MAXC>(Ra, Rb, gT, Gc, lane16);
                continue;
            }
            for (int side = 0; side < 2; ++side) {
                const RaRow &R = side ? Rb : Ra;
                if (R.n == -1) continue;
                float *orow = Gc + R.out;
                if (R.n >= 0) { ra_stream2<RA_MAXC>(R, R, gT, Gc, lane16); continue; }
                // stencil wider than 3 x 3 (beam voxels much coarser than patient voxels): plain loop over the candidate box
                for (int jj = lane16; jj < 4 * R.nq; jj += 16) {
                    const int j = R.j0 + jj;
                    float acc = 0.f;
                    for (int yy = R.ya; yy <= R.yb && j < P.Nv; ++yy) {
                        const float euy = R.eu0 + (yy - R.ya) * fu_y, ewy = R.ew0 + (yy - R.ya) * fw_y;
                        for (int xx = R.xa; xx <= R.xb; ++xx) {
                            const float wu = 1.f - fabsf(euy + (xx - R.xa) * fu_x), ww = 1.f - fabsf(ewy + (xx - R.xa) * fw_x);
                            if (wu > 0.f && ww > 0.f) acc = fmaf(wu * ww, __ldg(gT + ((size_t)yy * P.nx + xx) * nzp + j), acc);
                        }
                    }
                    orow[j] = acc;
                }
            }
        }
    }
}

// One pass of the convolution: sub-kernel (bi, bj) of the (NB KT)^2 window reads its inputs shifted by (su, sv) = ((bi, bj) - (NB-1)/2) KT:
//   out(i, j) (+)= sum_{di', dj' < KT} W_blk[di'][dj'] in(i + di' - c' + su, j + dj' - c' + sv),   c' = (KT-1)/2.
// The first pass (the centre block) writes every thread-tile of the output box, the others add to the tiles they reach.
struct ConvPass { int su, sv, first; };

// Geometry of one conv work item (control point, slice, chunk along v); identical in every lane of the warp.
struct ConvItem {
    int slot, cp, k;
    int pv, nts;
    long long slice_off;             // slot * stride_cp + k * pu * pv  (start of the [pu][pv] slice in the compact blocks)
    int ri0, rj0;
    SliceBox S, B, R;                // fluence support of the slice; source box of the input rows (S forward, F adjoint); outputs this pass reaches
    int ctf0, ctf1;                  // thread-tile range of the chunk along v
    int atf0, ats0, naf, nas;        // active thread-tiles of the slice and chunk (outputs to compute)
    int av0;                         // v index of the first active output column (forward: tile-aligned; adjoint: S.v0 & ~1)
    int n_tiles;                     // naf * nas
    int pitch, ring, tv0, tu0;       // input rows: pitch, rows the ring holds, input coords of window row 0 / column 0
    int n0;                          // slice kernel: table node and fraction
    float f;
};

template <int KT, bool ADJ, int CPL>
__device__ __forceinline__ void conv_load_item(const Params &P, const CpDesc *__restrict__ desc, int cp0, int n_cp,
                                               const int *__restrict__ tile_base, const float *__restrict__ zrad,
                                               const ConvPass &pass, int item, int &slot_hint, ConvItem &it)
{
    constexpr int C = (KT - 1) / 2;
    while (slot_hint + 1 < n_cp && item >= tile_base[slot_hint + 1]) ++slot_hint;   // items arrive in increasing order
    it.slot = slot_hint;
    it.cp = cp0 + it.slot;
    const CpDesc d = desc[it.cp];
    const int local = item - tile_base[it.slot];
    it.k = local / d.ncf;
    const int cf = local - it.k * d.ncf;
    it.ri0 = d.ri0; it.rj0 = d.rj0; it.pv = d.pv; it.nts = d.nts;
    it.slice_off = (long long)it.slot * P.stride_cp + (long long)it.k * d.pu * d.pv;
    it.ctf0 = cf * d.ntfc; it.ctf1 = min(d.ntf, it.ctf0 + d.ntfc);
    it.S = slice_support(P, d, it.k);
    const SliceBox F = dilate(P, it.S, P.CH);
    it.B = ADJ ? F : it.S;
    if (CPL == 2) { it.B.v0 &= ~1; it.B.v1 |= 1; }                // row copies move aligned pairs (k_project / k_resample_adjoint write them)
    // outputs this pass can reach: forward, the footprint of the shifted sub-kernel; adjoint, all of S_k (every input in F_k counts)
    it.R = ADJ ? it.S : F;
    if (!ADJ) {
        it.R.u0 = max(F.u0, it.S.u0 - pass.su - C); it.R.u1 = min(F.u1, it.S.u1 - pass.su + C);
        it.R.v0 = max(F.v0, it.S.v0 - pass.sv - C); it.R.v1 = min(F.v1, it.S.v1 - pass.sv + C);
        if (box_empty(it.S)) { it.R.u0 = 1; it.R.u1 = 0; }
    }
    const SliceBox A = ADJ ? it.S : (pass.first ? F : it.R);      // outputs to compute (the first pass also zero-fills what it does not reach)
    int atf0 = 0, atf1 = -1, ats0 = 0, ats1 = -1;
    if (!box_empty(A)) {
        atf0 = max(it.ctf0, (A.v0 - d.rj0) / RF); atf1 = min(it.ctf1 - 1, (A.v1 - d.rj0) / RF);
        ats0 = (A.u0 - d.ri0) / RS; ats1 = min(d.nts - 1, (A.u1 - d.ri0) / RS);
    }
    const bool any = atf0 <= atf1 && ats0 <= ats1;
    it.atf0 = atf0; it.ats0 = ats0; it.naf = any ? atf1 - atf0 + 1 : 0; it.nas = any ? ats1 - ats0 + 1 : 0;
    it.av0 = d.rj0 + atf0 * RF;
    if (ADJ && any && d.ncf == 1) {
        // adjoint outputs are read back only on S_k: start the thread-tiles at S.v0 (even, for the paired copies) instead of
        // the region's tile grid, which saves the partly used tile column at either end
        it.av0 = A.v0 & ~1;
        it.naf = (A.v1 - it.av0) / RF + 1;
    }
    it.n_tiles = it.naf * it.nas;
    it.pitch = conv_pitch(KT, max(it.naf, 1));
    it.ring = P.tile_floats / it.pitch;
    it.tv0 = it.av0 - C + pass.sv; it.tu0 = d.ri0 + ats0 * RS - C + pass.su;
    it.n0 = 0; it.f = 0.f;
    if (!any) return;
    // S4: slice kernel = lerp of the table in radiological depth
    const float t = zrad[(size_t)it.cp * P.Nw + it.k] / P.dz;
    int n0 = (int)floorf(t);
    n0 = min(max(n0, 0), P.n_z - 2);
    it.n0 = n0;
    it.f = fminf(fmaxf(t - n0, 0.f), 1.f);
}

// S4 + S5 (forward) / S8 (adjoint).  One WARP per block, many blocks per SM, persistent over the item list
// (control point, slice, chunk along v); items are handed out by a global counter.  A warp owns its input rows
// and its copy of the slice kernel in shared memory, so there is no block-level barrier anywhere.  It walks the
// active thread-tiles of its slice (F_k forward, S_k adjoint) in row-major order, 32 at a time (one 8(v) x 2(u)
// thread-tile per lane); the input rows live in a ring of shared-memory rows that slides down the slice, so every
// input row is fetched once per slice (cp.async in aligned pairs, zero-filled outside the source box: S_k
// forward, F_k adjoint), and geometry and slice kernel are worked out once per slice.  Slices are small (a few
// hundred thread-tiles): a block-wide tile shared through __syncthreads left the warps waiting on each other for
// almost half of their time (profiles/); independent warps balance by construction, and the other warps resident
// on the SM keep the FFMA pipe busy while one waits for its copies.
// CPL: floats per asynchronous copy, 2 when source and tile columns share parity ((C - sv) even).  MULTI: one of several passes
// (shifted sub-kernel: unreached tiles, accumulation into the output); the single-pass instance carries none of that code.
template <int KT, bool ADJ, int CPL, bool MULTI>
__global__ void __launch_bounds__(CONV_THREADS)
k_conv(Params P, const CpDesc *__restrict__ desc, int cp0, int n_cp, const int *__restrict__ tile_base,
       const float *__restrict__ zrad, const float *__restrict__ wtab, const float *__restrict__ in, float *__restrict__ out,
       int *item_counter, ConvPass pass)
{
    constexpr int KP = (KT + 3) & ~3;                 // weight row pitch [floats]
    constexpr int XW = (KT + RF - 1 + 3) & ~3;        // register window along v [floats]
    constexpr int NXQ = XW / 4;
    constexpr int PMAX = (NTFC_MAX * RF + XW - RF + 7) & ~7;   // widest row
    constexpr int MC = (PMAX / CPL + 31) / 32;        // copies per lane and row
    extern __shared__ float4 smem4[];
    // slice kernel as row pairs: Ws2[y][dj] = (W[y][dj], W[y-1][dj]), y = 0..KT, zero where the row does not exist — the two
    // weights an input row y contributes to the two output rows of a thread-tile, ready for one packed FFMA2
    float2 *Ws2 = reinterpret_cast<float2 *>(smem4);  // [(KT + 1) (du)][KP (dv)]
    float *tile = reinterpret_cast<float *>(smem4) + 2 * (KT + 1) * KP;   // ring of input rows [ring][pitch (v)]
    const unsigned tile_s = (unsigned)__cvta_generic_to_shared(tile);
    const int lane = threadIdx.x;
    const int total = tile_base[n_cp];
    int slot_hint = 0;

    for (;;) {
        int item = 0;
        if (lane == 0) item = atomicAdd(item_counter, 1);
        item = __shfl_sync(0xffffffffu, item, 0);
        if (item >= total) break;
        ConvItem I;
        conv_load_item<KT, ADJ, CPL>(P, desc, cp0, n_cp, tile_base, zrad, pass, item, slot_hint, I);
        float *oslice = out + I.slice_off;             // [pu][pv] of slice k
        if (I.n_tiles == 0) continue;                  // uniform across the warp
        const int pitch = I.pitch, ring = I.ring, naf = I.naf;
        {   // S4: slice kernel = lerp of the table in radiological depth; the table is stored as the [du][dv] image and is
            // point-symmetric, so forward and adjoint (flipped kernel) read the same entries
            const float *w0 = wtab + (size_t)I.n0 * KT * KP, *w1 = w0 + KT * KP;
            const float f = I.f;
            for (int e = lane; e < (KT + 1) * KP; e += 32) {
                const int y = e / KP;
                const float hi = y < KT ? (1.f - f) * __ldg(w0 + e) + f * __ldg(w1 + e) : 0.f;
                const float lo = y > 0 ? (1.f - f) * __ldg(w0 + e - KP) + f * __ldg(w1 + e - KP) : 0.f;
                Ws2[e] = make_float2(hi, lo);
            }
        }
        // column terms of the row copies (source offset, swizzled destination, validity): once per slice
        int joff[MC];
        unsigned doff[MC];
        bool cex[MC], cin[MC];
#pragma unroll
        for (int m = 0; m < MC; ++m) {
            const int c = CPL * (lane + 32 * m), j = I.tv0 + c;
            cex[m] = c < pitch;
            cin[m] = cex[m] && j >= I.B.v0 && j <= I.B.v1;                 // pairs are inside or outside as a whole (aligned box)
            joff[m] = cin[m] ? j - I.rj0 : 0;
            doff[m] = 4u * (unsigned)swz_col(c);
        }
        const float *sbase = in + I.slice_off;                             // row i of the slice at sbase + (i - ri0) * pv
        const float *tile_end = tile + ring * pitch;
        int loaded = 0;                                                    // window rows [0, loaded) have been fetched

        for (int t0 = 0; t0 < I.n_tiles; t0 += CONV_CHUNK_TILES) {
            const int ts_lo = t0 / naf, ts_hi = (min(I.n_tiles, t0 + CONV_CHUNK_TILES) - 1) / naf;
            const int need_lo = ts_lo * RS, need_hi = ts_hi * RS + RS - 1 + KT - 1;     // window rows of this group (inclusive)
            __syncwarp();                                                  // rows below need_lo are free to be overwritten
            {
                int w = max(loaded, need_lo), pos = w % ring;
                // per-lane source pointers and destination offsets advance by one row per iteration (no 64-bit
                // multiplies in the loop); rows outside the source box read nothing (size 0) from the slice start
                const float *sp[MC];
#pragma unroll
                for (int m = 0; m < MC; ++m) sp[m] = sbase + (long long)(I.tu0 + w - I.ri0) * I.pv + joff[m];
                unsigned drow = tile_s + 4u * (unsigned)(pos * pitch);
                const unsigned dstep = 4u * (unsigned)pitch, dend = tile_s + 4u * (unsigned)(ring * pitch);
                for (; w <= need_hi; ++w) {
                    const int i = I.tu0 + w;
                    const bool rin = i >= I.B.u0 && i <= I.B.u1;
#pragma unroll
                    for (int m = 0; m < MC; ++m) {
                        if (cex[m]) {
                            const bool ok = rin && cin[m];
                            if (CPL == 2) cp_async_8(drow + doff[m], ok ? sp[m] : sbase, ok ? 8 : 0);
                            else cp_async_4(drow + doff[m], ok ? sp[m] : sbase, ok ? 4 : 0);
                        }
                        sp[m] += I.pv;
                    }
                    drow += dstep;
                    if (drow == dend) drow = tile_s;
                }
                loaded = need_hi + 1;
            }
            cp_async_wait_all();
            __syncwarp();

            const int t = t0 + lane;
            if (t < I.n_tiles) {
                const int tsa = t / naf, tf = t - tsa * naf;
                static_assert(RS == 2, "the packed FFMA2 loop pairs the two output rows of a thread-tile");
                float2 acc2[RF];                   // (row 0, row 1) of output column r
#pragma unroll
                for (int r = 0; r < RF; ++r) acc2[r] = make_float2(0.f, 0.f);
                // forward: input rows outside S_k hold zeros (structurally zero fluence) and are skipped
                const int ylo = ADJ ? 0 : max(0, I.S.u0 - I.tu0 - tsa * RS), yhi = ADJ ? KT + RS - 2 : min(KT + RS - 2, I.S.u1 - I.tu0 - tsa * RS);
                // forward: a thread-tile that this pass's sub-kernel does not reach keeps its zeros (only the first pass has such tiles)
                const int ou = (I.ats0 + tsa) * RS + I.ri0, ov = I.av0 + tf * RF;
                const bool live = ADJ || !MULTI || (ou + RS - 1 >= I.R.u0 && ou <= I.R.u1 && ov + RF - 1 >= I.R.v0 && ov <= I.R.v1);
                const float *xrow = tile + ((tsa * RS + ylo) % ring) * pitch;
                int xoff[NXQ];
#pragma unroll
                for (int q = 0; q < NXQ; ++q) xoff[q] = swz_col(tf * RF + 4 * q);
                const float4 *w4 = reinterpret_cast<const float4 *>(Ws2 + ylo * KP);
#pragma unroll 1
                for (int y = live ? ylo : yhi + 1; y <= yhi; ++y) {
                    float2 xx[XW];                 // window element duplicated: it multiplies the weights of both output rows
#pragma unroll
                    for (int q = 0; q < NXQ; ++q) {
                        const float4 v = *reinterpret_cast<const float4 *>(xrow + xoff[q]);
                        xx[4 * q] = make_float2(v.x, v.x); xx[4 * q + 1] = make_float2(v.y, v.y);
                        xx[4 * q + 2] = make_float2(v.z, v.z); xx[4 * q + 3] = make_float2(v.w, v.w);
                    }
                    // one FFMA2 (fma.rn.f32x2) does the two multiply-adds of a tap for both output rows: half the issue
                    // slots of scalar FFMA, which leaves room for the LDS and address instructions beside a busy FMA pipe
#pragma unroll
                    for (int q = 0; q < KP / 2; ++q) {
                        const float4 wq4 = w4[q];
                        const float2 wq[2] = { make_float2(wq4.x, wq4.y), make_float2(wq4.z, wq4.w) };
#pragma unroll
                        for (int e = 0; e < 2; ++e) {
                            const int dj = 2 * q + e;
                            if (dj < KT) {
#pragma unroll
                                for (int r = 0; r < RF; ++r) acc2[r] = __ffma2_rn(xx[r + dj], wq[e], acc2[r]);
                            }
                        }
                    }
                    w4 += KP / 2;
                    xrow += pitch;
                    if (xrow == tile_end) xrow = tile;
                }
                float acc[RS][RF];
#pragma unroll
                for (int r = 0; r < RF; ++r) { acc[0][r] = acc2[r].x; acc[1][r] = acc2[r].y; }
#pragma unroll
                for (int ii = 0; ii < RS; ++ii) {
                    float *op = oslice + (size_t)((I.ats0 + tsa) * RS + ii) * I.pv + (I.av0 - I.rj0) + tf * RF;
                    if (ADJ) {                     // 8-byte aligned only; columns past the region are never read
                        const int room = I.pv - ((I.av0 - I.rj0) + tf * RF);
#pragma unroll
                        for (int r = 0; r < RF; r += 2)
                            if (r + 2 <= room) {
                                float2 *o = reinterpret_cast<float2 *>(op + r);
                                float2 v = make_float2(acc[ii][r], acc[ii][r + 1]);
                                if (MULTI && !pass.first) { const float2 p = *o; v.x += p.x; v.y += p.y; }
                                *o = v;
                            }
                    } else {
                        float4 *o = reinterpret_cast<float4 *>(op);
                        float4 v0 = make_float4(acc[ii][0], acc[ii][1], acc[ii][2], acc[ii][3]), v1 = make_float4(acc[ii][4], acc[ii][5], acc[ii][6], acc[ii][7]);
                        if (MULTI && !pass.first) {
                            const float4 p0 = o[0], p1 = o[1];
                            v0.x += p0.x; v0.y += p0.y; v0.z += p0.z; v0.w += p0.w; v1.x += p1.x; v1.y += p1.y; v1.z += p1.z; v1.w += p1.w;
                        }
                        o[0] = v0; o[1] = v1;
                    }
                }
            }
        }
        __syncwarp();                                  // the next item overwrites the rows and the slice kernel
    }
}

// Expands the compact block of one control point to a dense [Nw][Nv][Nu] volume (stage tap for tests).
__global__ void k_expand_dense(Params P, const CpDesc *__restrict__ desc, const SliceBox16 *__restrict__ wbox, int cp, int slot,
                               const float *__restrict__ comp, float *__restrict__ dense)
{
    const CpDesc d = desc[cp];
    const size_t n = (size_t)P.Nu * P.Nv * P.Nw;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const int i = (int)(e % P.Nu), j = (int)((e / P.Nu) % P.Nv), k = (int)(e / ((size_t)P.Nu * P.Nv));
        float v = 0.f;
        if (d.a0 <= d.a1) {                      // outside the written box of the slice the block holds stale data: D_b is zero there
            const SliceBox16 w = load_box(wbox, (size_t)cp * P.Nw + k);
            if (i >= w.u0 && i <= w.u1 && j >= w.v0 && j <= w.v1) v = comp[compact_index(P, d, slot, i, j, k)];
        }
        dense[e] = v;
    }
}

// dL/dDose [nz][ny][nx] -> gT [ny*nx][nzp] (z fastest, row pitch nzp = nz rounded up to 4, pad zero), 32x32
// shared-memory tiles.  Grid: (ceil(nxy/32), ceil(nzp/32)).
__global__ void __launch_bounds__(256) k_transpose_g(int nxy, int nz, int nzp, const float *__restrict__ g, float *__restrict__ gT)
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
        if (p < nxy && z < nzp) gT[(size_t)p * nzp + z] = t[lx][r];
    }
}

}  // namespace pdrt
