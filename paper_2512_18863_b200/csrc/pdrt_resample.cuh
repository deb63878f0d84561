// pdrt_resample.cuh — S6 (beam -> patient resampling + MU-weighted accumulation, PAPER.md:160-168,
// Eq. 9) and S9 (transpose of the divergent projection, Eq. 5-6, in gather form).  These are the
// bandwidth-bound stages: each patient voxel is written once per call (accumulation over control points
// stays in registers), the compact D_b / H_b blocks are read once as 16-byte vectors along v, and no global
// atomics are used anywhere.  (S7, the transpose of S6, is k_resample_adjoint in pdrt_conv.cuh.)
#pragma once
#include <cooperative_groups.h>

#include "pdrt_dev.cuh"

namespace pdrt {

namespace cg = cooperative_groups;

constexpr int GD_PX = 8, GD_PY = 4;              // a block owns 8 x 4 patient columns (x,y): 32-byte runs of the dose rows
constexpr int GD_COLS = GD_PX * GD_PY;
constexpr int GD_LANES = 8;                      // lanes per column: a quarter-warp reads 128 contiguous bytes of a beam row.  Every lane
                                                 // of a column fetches the column's stencil record from shared memory, and a warp-wide
                                                 // LDS.128 takes four data-pipe cycles however many lanes share an address: with 8 lanes
                                                 // instead of 16 the records cost half as many cycles per byte of D_b
constexpr int GD_CPB = 8;                        // control points set up per round (32 columns x 8 control points = 256 threads)
constexpr int GD_THREADS = GD_COLS * GD_CPB;
static_assert(GD_THREADS == GD_COLS * GD_LANES, "phase A (column, control point) and phase B (column, lane) use the same threads");
constexpr int GD_ZSPAN = 4 * GD_LANES;           // z covered by one pass of a column's lanes (8 lanes x float4)
constexpr int GD_MAXPASS = 4;                    // passes held in registers at once (128 z)
constexpr int GD_LIST = GD_THREADS;              // control points listed per outer chunk: one thread each

struct __align__(16) GatherCp {                  // what the stencil set-up needs of a listed control point (32 bytes, shared memory)
    float cg, sg, scale;
    int ri0, pu, pv, rj0, slot;
};
struct __align__(16) GatherRec {                 // bilinear stencil of one (patient column, control point): 64 bytes in four 16-byte chunks
    ulonglong2 q[4];                             // chunk c sits at q[c ^ gather_swz(column)]: the records of consecutive columns are 64 bytes
                                                 // apart, and unswizzled their chunks would fall on two bank groups (4-way conflicts
                                                 // of the set-up's stores)
    // chunk 0: beam rows (i0,k0), (i0+1,k0); chunk 1: rows (i0,k0+1), (i0+1,k0+1) — pointers shifted so that row[z] is voxel v = z,
    //          invalid neighbours folded onto a valid row
    // chunk 2: four floats cal * MU * bilinear weight, 0 for invalid neighbours
    // chunk 3: .x = four shorts zlo0, zhi0, zlo1, zhi1: written v-range [zlo, zhi) of slice k0 and of slice k0+1 (multiples of 8);
    //          empty: no reads
};
__device__ __forceinline__ int gather_swz(int column) { return (column >> 1) & 3; }

// phase B of k_gather_dose for one round of control points: NP z-passes of 32 held in registers, NB control points per
// batch.  Straight-line code: the 4 NB NP loads of a batch are all issued before the first use.  Records of control points that
// do not reach the column carry empty z-ranges (no reads) and zero weights.
template <int NP, int NB>
__device__ __forceinline__ void gather_round(const GatherRec (*rec)[GD_COLS], int col, int nround, int zq, float2 (&acc)[GD_MAXPASS][2])
{
    const int sw = gather_swz(col);
    for (int e0 = 0; e0 < nround; e0 += NB) {
        float4 v[NB][NP][4];
        float4 w[NB];
#pragma unroll
        for (int q = 0; q < NB; ++q) {
            const GatherRec &R = rec[e0 + q][col];
            const int2 zr = *reinterpret_cast<const int2 *>(&R.q[3 ^ sw]);
            w[q] = *reinterpret_cast<const float4 *>(&R.q[2 ^ sw]);
            const int zlo0 = (short)(zr.x & 0xffff), zhi0 = zr.x >> 16, zlo1 = (short)(zr.y & 0xffff), zhi1 = zr.y >> 16;
            const ulonglong2 ra = R.q[sw], rb = R.q[1 ^ sw];
            const float *r0 = reinterpret_cast<const float *>(ra.x), *r1 = reinterpret_cast<const float *>(ra.y);
            const float *r2 = reinterpret_cast<const float *>(rb.x), *r3 = reinterpret_cast<const float *>(rb.y);
#pragma unroll
            for (int ps = 0; ps < NP; ++ps) {
                const int z = zq + ps * GD_ZSPAN;
                const bool in0 = z >= zlo0 && z < zhi0, in1 = z >= zlo1 && z < zhi1;
                const float4 zero = make_float4(0.f, 0.f, 0.f, 0.f);
                v[q][ps][0] = in0 ? __ldg(reinterpret_cast<const float4 *>(r0 + z)) : zero;
                v[q][ps][1] = in0 ? __ldg(reinterpret_cast<const float4 *>(r1 + z)) : zero;
                v[q][ps][2] = in1 ? __ldg(reinterpret_cast<const float4 *>(r2 + z)) : zero;
                v[q][ps][3] = in1 ? __ldg(reinterpret_cast<const float4 *>(r3 + z)) : zero;
            }
        }
#pragma unroll
        for (int q = 0; q < NB; ++q) {                       // control-point order (deterministic); packed FFMA2: two z per instruction
            const float wq[4] = { w[q].x, w[q].y, w[q].z, w[q].w };
#pragma unroll
            for (int ps = 0; ps < NP; ++ps)
#pragma unroll
                for (int n = 0; n < 4; ++n) {
                    const float2 w2 = make_float2(wq[n], wq[n]);
                    acc[ps][0] = __ffma2_rn(w2, make_float2(v[q][ps][n].x, v[q][ps][n].y), acc[ps][0]);
                    acc[ps][1] = __ffma2_rn(w2, make_float2(v[q][ps][n].z, v[q][ps][n].w), acc[ps][1]);
                }
        }
    }
}

// S6.  Grid: (ceil(nx/8), ceil(ny/4), 1); a block owns 8 x 4 patient columns (x,y) over all z.
//   dose[p] (+)= sum_b scale_b * bilinear_0(D_b[.][z][.]; fu, fw)
// The gantry rotates about z (G1), so for one control point the beam-frame position (fu, fw) and the four
// bilinear weights of a column are the same for all its voxels.  Warp 0 first lists the control points whose compact
// region can reach the block's columns (with the constants the set-up needs, and the z-range they cover).  Then, 8
// control points at a time: phase A, one THREAD per (column, control point) builds the stencil record (pointers to the four
// beam rows, weights, and the v-range that the forward conv wrote in the two slices — outside it D_b is zero and the block
// holds stale data); phase B, one QUARTER-WARP per column streams 16-byte vectors along v, several control points per batch
// with all their loads in flight at once, accumulating in registers in control-point order (deterministic).  The records
// are double-buffered and the global reads of phase A for round r+1 are issued before phase B of round r, so that their
// latency is covered.  Every patient voxel of the z-range is written exactly once; the rest of the dose grid is zeroed by
// the caller (memset).
__global__ void __launch_bounds__(GD_THREADS, 2)
k_gather_dose(Params P, const CpDesc *__restrict__ desc, const SliceBox16 *__restrict__ wbox, int cp0, int n_cp,
              const float *__restrict__ D, float *__restrict__ dose, int accumulate)
{
    __shared__ GatherRec rec[2][GD_CPB][GD_COLS];
    __shared__ GatherCp list[GD_LIST];
    __shared__ int n_list_s, zmin_s, zmax_s, wcount_s[GD_THREADS / 32], wzlo_s[GD_THREADS / 32], wzhi_s[GD_THREADS / 32];
    const int tid = threadIdx.x, lz = tid & (GD_LANES - 1);
    const int col = tid / GD_LANES;                              // phase B: column of this quarter-warp
    const int a_col = tid & (GD_COLS - 1), a_cp = tid / GD_COLS; // phase A: (column, control point of the round)
    const int px0 = blockIdx.x * GD_PX, py0 = blockIdx.y * GD_PY;
    // tile corners (for culling), relative to the isocentre
    const float cx0 = P.ox + px0 * P.sx - P.isox, cx1 = cx0 + (GD_PX - 1) * P.sx;
    const float cy0 = P.oy + py0 * P.sy - P.isoy, cy1 = cy0 + (GD_PY - 1) * P.sy;
    // phase-A column of this thread
    const int ax = px0 + (a_col & (GD_PX - 1)), ay = py0 + a_col / GD_PX;
    const float adx = P.ox + ax * P.sx - P.isox, ady = P.oy + ay * P.sy - P.isoy;
    const bool a_inside = ax < P.nx && ay < P.ny;
    // phase-B column of this quarter-warp
    const int bx = px0 + (col & (GD_PX - 1)), by = py0 + col / GD_PX;
    const bool b_inside = bx < P.nx && by < P.ny;

    // phase A, first half: position of the column in the beam frame of control point list[q]; issues the reads of the two slice boxes
    struct Setup { int i0, k0; float tu, tw; SliceBox16 w0, w1; bool on; };
    auto setup_load = [&](int q, int n_list) {
        Setup s;
        s.on = q < n_list && a_inside;
        s.w0 = SliceBox16{ 1, 0, 1, 0 }; s.w1 = s.w0;
        s.i0 = s.k0 = 0; s.tu = s.tw = 0.f;
        if (s.on) {
            const GatherCp g = list[q];
            const float fu = (g.cg * adx + g.sg * ady) / P.du + P.cu;
            const float fw = (-g.sg * adx + g.cg * ady - P.wmin) / P.dw;
            const float flu = floorf(fu), flw = floorf(fw);
            s.i0 = (int)flu; s.k0 = (int)flw;
            s.tu = fu - flu; s.tw = fw - flw;
            // bilinear_0: neighbours outside the beam grid contribute 0; outside the written box of its slice D_b is 0
            const size_t base = (size_t)(cp0 + g.slot) * P.Nw;
            if (s.k0 >= 0 && s.k0 < P.Nw) s.w0 = load_box(wbox, base + s.k0);
            if (s.k0 + 1 >= 0 && s.k0 + 1 < P.Nw) s.w1 = load_box(wbox, base + s.k0 + 1);
        }
        return s;
    };
    // phase A, second half: the record
    auto setup_store = [&](const Setup &s, int q, GatherRec &R) {
        bool v00 = false, v10 = false, v01 = false, v11 = false;
        if (s.on) {
            v00 = s.i0 >= s.w0.u0 && s.i0 <= s.w0.u1; v10 = s.i0 + 1 >= s.w0.u0 && s.i0 + 1 <= s.w0.u1;
            v01 = s.i0 >= s.w1.u0 && s.i0 <= s.w1.u1; v11 = s.i0 + 1 >= s.w1.u0 && s.i0 + 1 <= s.w1.u1;
        }
        const float *row[4] = { D, D, D, D };
        float4 wv = make_float4(0.f, 0.f, 0.f, 0.f);
        short zlo0 = 0, zhi0 = 0, zlo1 = 0, zhi1 = 0;
        if (v00 || v10 || v01 || v11) {
            const GatherCp g = list[q];
            const int rs = g.pv, ks = g.pu * g.pv;
            const int o00 = (s.k0 * g.pu + (s.i0 - g.ri0)) * rs;
            const int any_off = v00 ? o00 : (v10 ? o00 + rs : (v01 ? o00 + ks : o00 + ks + rs));
            const float *base = D + (size_t)g.slot * (size_t)P.stride_cp - g.rj0;
            row[0] = base + (v00 ? o00 : any_off); row[1] = base + (v10 ? o00 + rs : any_off);
            row[2] = base + (v01 ? o00 + ks : any_off); row[3] = base + (v11 ? o00 + ks + rs : any_off);
            wv.x = v00 ? g.scale * ((1.f - s.tu) * (1.f - s.tw)) : 0.f; wv.y = v10 ? g.scale * (s.tu * (1.f - s.tw)) : 0.f;
            wv.z = v01 ? g.scale * ((1.f - s.tu) * s.tw) : 0.f; wv.w = v11 ? g.scale * (s.tu * s.tw) : 0.f;
            // a slice none of whose rows is valid gets an empty z-range: its (folded) rows are not read at all
            if (v00 || v10) { zlo0 = s.w0.v0; zhi0 = (short)(s.w0.v1 + 1); }
            if (v01 || v11) { zlo1 = s.w1.v0; zhi1 = (short)(s.w1.v1 + 1); }
        }
        const int sw = gather_swz(a_col);
        R.q[sw] = make_ulonglong2((unsigned long long)row[0], (unsigned long long)row[1]);
        R.q[1 ^ sw] = make_ulonglong2((unsigned long long)row[2], (unsigned long long)row[3]);
        *reinterpret_cast<float4 *>(&R.q[2 ^ sw]) = wv;
        *reinterpret_cast<int4 *>(&R.q[3 ^ sw]) = make_int4((int)(unsigned short)zlo0 | ((int)zhi0 << 16), (int)(unsigned short)zlo1 | ((int)zhi1 << 16), 0, 0);
    };

    for (int c0 = 0; c0 < n_cp; c0 += GD_LIST) {
        __syncthreads();
        {   // the ordered list of candidate control points and their z-range: one thread per control point of the chunk (GD_LIST = the
            // block size), kept entries compacted in control-point order by a ballot per warp and a prefix over the warps
            const int c = c0 + tid;
            bool keep = false;
            GatherCp g;
            int zlo = P.nz, zhi = 0;
            if (c < n_cp) {
                const CpDesc &d = desc[cp0 + c];
                if (d.a0 <= d.a1) {
                    g.cg = d.cg; g.sg = d.sg; g.scale = d.scale; g.ri0 = d.ri0; g.pu = d.pu; g.pv = d.pv; g.rj0 = d.rj0; g.slot = c;
                    // u-extent of the tile: extremes are at its corners
                    const float u00 = g.cg * cx0 + g.sg * cy0, u10 = g.cg * cx1 + g.sg * cy0;
                    const float u01 = g.cg * cx0 + g.sg * cy1, u11 = g.cg * cx1 + g.sg * cy1;
                    const float umin = fminf(fminf(u00, u10), fminf(u01, u11)) / P.du + P.cu;
                    const float umax = fmaxf(fmaxf(u00, u10), fmaxf(u01, u11)) / P.du + P.cu;
                    keep = umax >= (float)(g.ri0 - 1) && umin <= (float)(g.ri0 + g.pu);
                    if (keep) { zlo = g.rj0; zhi = min(P.nz, g.rj0 + g.pv); }
                }
            }
            const int lane = tid & 31, warp = tid >> 5;
            const unsigned m = __ballot_sync(0xffffffffu, keep);
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                zlo = min(zlo, __shfl_xor_sync(0xffffffffu, zlo, o));
                zhi = max(zhi, __shfl_xor_sync(0xffffffffu, zhi, o));
            }
            if (lane == 0) { wcount_s[warp] = __popc(m); wzlo_s[warp] = zlo; wzhi_s[warp] = zhi; }
            __syncthreads();
            int base = 0, total = 0, zmin = P.nz, zmax = 0;
#pragma unroll
            for (int w = 0; w < GD_THREADS / 32; ++w) {
                if (w < warp) base += wcount_s[w];
                total += wcount_s[w]; zmin = min(zmin, wzlo_s[w]); zmax = max(zmax, wzhi_s[w]);
            }
            if (keep) list[base + __popc(m & ((1u << lane) - 1u))] = g;
            if (tid == 0) { n_list_s = total; zmin_s = zmin & ~7; zmax_s = zmax; }
        }
        __syncthreads();
        const int n_list = n_list_s, zmin = zmin_s, zmax = zmax_s;
        if (n_list == 0) continue;
        for (int zb = zmin; zb < zmax; zb += GD_ZSPAN * GD_MAXPASS) {            // one iteration unless the regions span > 128 z
            float2 acc[GD_MAXPASS][2];                                           // [pass][z pair] of this lane's quads
#pragma unroll
            for (int p = 0; p < GD_MAXPASS; ++p) acc[p][0] = acc[p][1] = make_float2(0.f, 0.f);
            const int npass = min(GD_MAXPASS, (zmax - zb + GD_ZSPAN - 1) / GD_ZSPAN);
            const int zq = zb + 4 * lz;
            {   // records of round 0
                const Setup s = setup_load(a_cp, n_list);
                setup_store(s, a_cp, rec[0][a_cp][a_col]);
            }
            __syncthreads();
            int buf = 0;
            for (int q0 = 0; q0 < n_list; q0 += GD_CPB, buf ^= 1) {
                const Setup s = setup_load(q0 + GD_CPB + a_cp, n_list);          // reads for the next round are in flight during phase B
                const int nround = min(GD_CPB, n_list - q0);
                if (b_inside) {
                    if (npass == 1) gather_round<1, 4>(rec[buf], col, nround, zq, acc);
                    else if (npass == 2) gather_round<2, 2>(rec[buf], col, nround, zq, acc);
                    else gather_round<GD_MAXPASS, 1>(rec[buf], col, nround, zq, acc);
                }
                setup_store(s, q0 + GD_CPB + a_cp, rec[buf ^ 1][a_cp][a_col]);
                __syncthreads();
            }
            if (b_inside) {
#pragma unroll
                for (int ps = 0; ps < GD_MAXPASS; ++ps) {
                    if (ps >= npass) continue;
                    const int z = zb + ps * GD_ZSPAN + 4 * lz;
                    const float v[4] = { acc[ps][0].x, acc[ps][0].y, acc[ps][1].x, acc[ps][1].y };
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        if (z + e < zmax) {
                            float *o = dose + ((size_t)(z + e) * P.ny + by) * P.nx + bx;
                            *o = (accumulate || c0 > 0) ? *o + v[e] : v[e];
                        }
                    }
                }
            }
        }
    }
}

// S9.  gPhimap_b[pix] = sum_k mag_k^2 sum_{voxels} weight(voxel -> pix) * H_b[voxel]  in gather form.  The bilinear weight
// is separable, weight = wa(i; a, k) * wb(j; b, k).  A warp owns 32 pixel rows b of the fluence support bbox (lanes: b, the
// contiguous axis of H_b) and ALL pixel columns a.  Per slice it walks the voxel rows i of S_k once, in increasing i:
// each lane contracts its (at most 4) voxels along v, t = sum_j wb H[k][i][j] (coalesced), and the row adds (1-ta) t to
// pixel column a(i) and ta t to a(i)+1.  Since a(i) never decreases along the walk, two running sums suffice; a finished
// column is added to the warp's private plane in shared memory.  The slices of a control point are dealt round-robin to
// the 32 warps of a CLUSTER of four blocks; the planes are reduced in a fixed order, first inside each block, then across
// the cluster through distributed shared memory (deterministic, no atomics).
// Grid: (4 * ceil(Nvf/32), n_cp), cluster (4,1,1); dynamic shared memory n_act * Nuf * 32 floats.
constexpr int PA_THREADS = 256, PA_WARPS = PA_THREADS / 32, PA_CLUSTER = 4, PA_TAPS = 4, PA_ROWS = 4;

__global__ void __cluster_dims__(PA_CLUSTER, 1, 1) __launch_bounds__(PA_THREADS, 3)
k_project_adjoint(Params P, const CpDesc *__restrict__ desc, const SliceBox16 *__restrict__ sbox, int cp0, int n_cp, int n_act,
                  const float *__restrict__ H, float *__restrict__ gphimap)
{
    extern __shared__ float pa_smem[];                  // [n_act][bw][32]: n_act <= PA_WARPS warps work (very wide maps: fewer planes fit)
    cg::cluster_group cluster = cg::this_cluster();
    const int crank = (int)cluster.block_rank(), bchunk = blockIdx.x / PA_CLUSTER;
    const int slot = blockIdx.y;
    const int cp = cp0 + slot;
    const CpDesc d = desc[cp];
    // every block of a cluster shares (cp, bchunk): the early exits are taken by the whole cluster
    if (d.a0 > d.a1) return;
    const int B0 = d.pb0 + 32 * bchunk;
    if (B0 > d.pb1) return;
    const int bw = d.pa1 - d.pa0 + 1;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    float *plane = pa_smem + (size_t)min(warp, n_act - 1) * bw * 32;
    if (warp < n_act)
        for (int e = lane; e < bw * 32; e += 32) plane[e] = 0.f;
    __syncwarp();
    const int b = B0 + lane;
    const bool live = b <= d.pb1;
    const float *Hc = H + (size_t)slot * (size_t)P.stride_cp;
    const float vb = P.v0 / P.dv;                       // v_j / dv = vb + j
    for (int k = warp < n_act ? crank * n_act + warp : P.Nw; k < P.Nw; k += PA_CLUSTER * n_act) {
        const SliceBox16 S = load_box(sbox, (size_t)cp * P.Nw + k);
        if (S.u0 > S.u1) continue;
        const float mag = P.sid / (P.sid + P.wmin + k * P.dw), m2 = mag * mag;
        const float su = mag * P.du / P.Du, sv = mag * P.dv / P.Dv, iv = P.Dv / (mag * P.dv);
        // voxels with a non-zero weight onto pixel row b: fb(j) in the OPEN interval (b-1, b+1), at most 2 iv + 1 of them
        int jlo = max((int)S.v0, (int)floorf((b - 1 - P.cvf) * iv - vb) + 1), jhi = min((int)S.v1, (int)ceilf((b + 1 - P.cvf) * iv - vb) - 1);
        if (!live) jhi = jlo - 1;
        // v weights of this lane's (at most PA_TAPS) voxels, once per slice, times mag^2; wider stencils (beam voxels much finer
        // than the map pixels) take the general loop
        const bool few = __all_sync(0xffffffffu, jhi - jlo < PA_TAPS);
        float wbq[PA_TAPS];
#pragma unroll
        for (int e = 0; e < PA_TAPS; ++e) {
            const float wb = 1.f - fabsf((vb + jlo + e) * sv + P.cvf - (float)b);
            wbq[e] = (jlo + e <= jhi && wb > 0.f) ? m2 * wb : 0.f;
        }
        // per-lane row pointer at its first tap (a lane without taps reads column S.v0 with weight 0: every address is readable)
        const int jfirst = jlo <= jhi ? jlo : (int)S.v0;
        const float *hrow = Hc + ((size_t)k * d.pu + (S.u0 - d.ri0)) * d.pv - d.rj0 + jfirst;      // row S.u0; rows are d.pv apart
        const int ntap = few ? min(PA_TAPS, (int)S.v1 - jfirst + 1) : 0;                           // taps that stay inside the row
        int a_cur = (int)floorf((S.u0 - P.cu) * su + P.cuf);                                       // warp-uniform
        float acc_lo = 0.f, acc_hi = 0.f;
        for (int i = S.u0; i <= S.u1; i += PA_ROWS) {
            float t[PA_ROWS];
            if (few) {
                // straight-line: the PA_ROWS x PA_TAPS loads are all issued before the first use (rows past S.u1 re-read row S.u1)
                float hv[PA_ROWS][PA_TAPS];
#pragma unroll
                for (int r = 0; r < PA_ROWS; ++r) {
                    const float *h = hrow + (size_t)min(r, (int)S.u1 - i) * d.pv;
#pragma unroll
                    for (int e = 0; e < PA_TAPS; ++e) hv[r][e] = __ldg(h + (e < ntap ? e : 0));
                }
#pragma unroll
                for (int r = 0; r < PA_ROWS; ++r) {
                    t[r] = 0.f;
#pragma unroll
                    for (int e = 0; e < PA_TAPS; ++e) t[r] = fmaf(wbq[e], hv[r][e], t[r]);
                }
            } else {
#pragma unroll
                for (int r = 0; r < PA_ROWS; ++r) {
                    t[r] = 0.f;
                    if (i + r <= S.u1) {
                        const float *h = hrow + (size_t)r * d.pv - jfirst;
                        for (int j = jlo; j <= jhi; ++j) {
                            const float wb = 1.f - fabsf((vb + j) * sv + P.cvf - (float)b);
                            if (wb > 0.f) t[r] = fmaf(m2 * wb, __ldg(h + j), t[r]);
                        }
                    }
                }
            }
            hrow += (size_t)PA_ROWS * d.pv;
#pragma unroll
            for (int r = 0; r < PA_ROWS; ++r) {
                if (i + r > S.u1) break;
                const float fa = (i + r - P.cu) * su + P.cuf;
                const float fla = floorf(fa);
                const int a0 = (int)fla;
                const float ta = fa - fla;
                while (a_cur < a0) {                      // column a_cur is complete (a(i) never decreases): warp-uniform
                    if (a_cur >= d.pa0 && a_cur <= d.pa1) plane[(a_cur - d.pa0) * 32 + lane] += acc_lo;
                    acc_lo = acc_hi; acc_hi = 0.f; ++a_cur;
                }
                acc_lo = fmaf(1.f - ta, t[r], acc_lo);
                acc_hi = fmaf(ta, t[r], acc_hi);
            }
        }
        if (a_cur >= d.pa0 && a_cur <= d.pa1) plane[(a_cur - d.pa0) * 32 + lane] += acc_lo;
        if (a_cur + 1 >= d.pa0 && a_cur + 1 <= d.pa1) plane[(a_cur + 1 - d.pa0) * 32 + lane] += acc_hi;
    }
    __syncthreads();
    // the block's warps, in warp order, into plane 0
    for (int e = tid; e < bw * 32; e += PA_THREADS) {
        float s = 0.f;
        for (int w = 0; w < n_act; ++w) s += pa_smem[(size_t)w * bw * 32 + e];
        pa_smem[e] = s;
    }
    cluster.sync();
    // the cluster's blocks, in rank order; block r writes the pixels e = r, r + 4, ... (a fastest in gphimap)
    const float *remote[PA_CLUSTER];
#pragma unroll
    for (int q = 0; q < PA_CLUSTER; ++q) remote[q] = cluster.map_shared_rank(pa_smem, q);
    for (int t = crank * PA_THREADS + tid; t < bw * 32; t += PA_CLUSTER * PA_THREADS) {
        const int a = t % bw, bl = t / bw;               // consecutive threads: consecutive a
        float s = 0.f;
#pragma unroll
        for (int q = 0; q < PA_CLUSTER; ++q) s += remote[q][a * 32 + bl];
        if (B0 + bl <= d.pb1) gphimap[((size_t)cp * P.Nvf + B0 + bl) * P.Nuf + d.pa0 + a] = s;
    }
    cluster.sync();                                      // nobody leaves while its shared memory is still being read
}

}  // namespace pdrt
