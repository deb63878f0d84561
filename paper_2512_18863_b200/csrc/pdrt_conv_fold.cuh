// pdrt_conv_fold.cuh — the row-symmetric convolution of pdrt_conv_sym.cuh with the kernel's COLUMN symmetry folded in as well
// (the pencil kernel is radially symmetric; R3: the table is built mirrored in both axes).
//
// A row correlation is  T_d[r][j] = W_d[C] x[r][j] + sum_{m=1..C} W_d[C+m] (x[r][j-m] + x[r][j+m]),  W_d = row C+d of the slice
// kernel.  The folded window  z[j][m] = x[r][j-m] + x[r][j+m]  does not depend on d: a unit = (row pair r, r+1) x W output columns
// (W = 4 up to 31 taps, 2 above) builds its W x (C+1) folded values once (packed adds on the (row r, row r+1) pairs) and then runs the C+1 steps d = C .. 0 with
// C+1 packed FFMA2 per column instead of 2C+1.  Together with the row symmetry that is (C+1)^2 multiply-adds per input value
// instead of (2C+1)^2.  Everything else is pdrt_conv_sym.cuh: one warp per block, units of 32 lanes, output rows accumulated in a
// warp-private shared-memory ring (one 16- or 8-byte read-modify-write per side and step), staged input rows, rows written to HBM
// when no later unit reaches them.  The folded window takes 2 W (C+2) registers.
#pragma once
#include "pdrt_conv_sym.cuh"

namespace pdrt {

constexpr int FOLD_COLS_MAX = 8 * SYM_NTFC_MAX;     // widest work item [columns]
// from 55 taps the work items are at most 48 columns wide: the ring of 2 C + 2 maxp output rows is what fills the shared memory there
// (measured on c4, forward / backward of the whole call: 63 taps 9.58 / 7.91 -> 9.00 / 7.18 ms, 75 taps 14.5 / 11.4 -> 12.9 / 9.8 ms)
__host__ __device__ constexpr int fold_cols_max(int kt) { return kt >= 55 ? 48 : FOLD_COLS_MAX; }
// output columns per unit: 4 up to 31 taps, 2 above (the folded window takes 2 W (C + 2) registers)
__host__ __device__ constexpr int fold_unit_cols(int kt) { return kt <= 31 ? 4 : 2; }

// ring row pitch [floats] for nt units of w columns.  Units of 4 columns: one 16-byte chunk per unit, padded until the chunks of
// the next row pair (two rows on) continue where this row ends, give or take one chunk (modulo the 8 chunks of a wavefront).
__host__ __device__ __forceinline__ int fold_out_pitch(int nt, int w)
{
    if (w != 4) return (w * nt + 3) & ~3;
    for (int p = 4 * nt;; p += 4) {
        const int dl = (p >> 1) & 7;
        if (dl == (nt & 7) || dl == ((nt + 1) & 7) || dl == ((nt - 1) & 7)) return p;
    }
}
__host__ __device__ __forceinline__ int fold_max_pairs(int nt) { return (30 + nt) / nt + 1 < 8 ? (30 + nt) / nt + 1 : 8; }
// 16-byte chunks (2 columns x 2 rows) per staged row pair (even: the swizzle swaps neighbours)
__host__ __device__ __forceinline__ int fold_in_chunks(int nt, int w, int c) { return ((w * nt + 2 * c) / 2 + 1) & ~1; }
inline int fold_out_floats(int kt)
{
    const int c = (kt - 1) / 2, w = fold_unit_cols(kt);
    int best = 0;
    for (int n = 1; n <= fold_cols_max(kt) / w; ++n) best = std::max(best, (2 * fold_max_pairs(n) + 2 * c) * fold_out_pitch(n, w));
    return best;
}
inline int fold_in_floats(int kt)
{
    const int c = (kt - 1) / 2, w = fold_unit_cols(kt);
    int best = 0;
    for (int n = 1; n <= fold_cols_max(kt) / w; ++n) best = std::max(best, fold_max_pairs(n) * fold_in_chunks(n, w, c) * 4);
    return best;
}
__host__ __device__ constexpr int fold_wpitch(int kt) { return ((kt - 1) / 2 + 1 + 3) & ~3; }         // floats per weight row: W_d[C .. 2C], padded to 4
inline size_t fold_smem_bytes(int kt)
{
    const int c = (kt - 1) / 2;
    return sizeof(float) * ((size_t)(c + 1) * fold_wpitch(kt) + fold_in_floats(kt) + fold_out_floats(kt));
}

// 16- / 8-byte accesses of the ring by shared-window address (an address register per row instead of a generic pointer whose
// window base the compiler would re-derive from the special registers in every step)
__device__ __forceinline__ float4 ring_ld4(unsigned a)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void ring_st4(unsigned a, const float4 &v)
{
    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(a), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ float2 ring_ld2(unsigned a)
{
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void ring_st2(unsigned a, const float2 &v)
{
    asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(a), "f"(v.x), "f"(v.y) : "memory");
}

// One step d of a unit: acc = (a_d, b_d) from the folded window and the weight row in `w`; then the next step's weights are fetched
// and out[r-d] += a_d + b_{d+1}, out[r+1+d] += b_d + a_{d+1} with (a_{d+1}, b_{d+1}) = prev.  om / op: shared-window addresses of the
// unit's columns in the two ring rows; hm / hp: whether the row is held.
template <int C, int FRF>
__device__ __forceinline__ void fold_step(const float2 (&zc)[FRF], const float2 (&z)[C][FRF], float4 (&w)[(C + 4) / 4], const float4 *__restrict__ wnext,
                                          float2 (&acc)[FRF], const float2 (&prev)[FRF], unsigned om, bool hm, unsigned op, bool hp)
{
    constexpr int WQ = (C + 4) / 4;
#pragma unroll
    for (int q = 0; q < WQ; ++q) {
        const float ws[4] = { w[q].x, w[q].y, w[q].z, w[q].w };
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int m = 4 * q + e;
            if (m <= C) {
                const float2 wd = make_float2(ws[e], ws[e]);          // one register: FFMA2 takes it as a scalar operand
#pragma unroll
                for (int c = 0; c < FRF; ++c) acc[c] = m == 0 ? __fmul2_rn(zc[c], wd) : __ffma2_rn(z[m - 1][c], wd, acc[c]);
            }
        }
    }
#pragma unroll
    for (int q = 0; q < WQ; ++q) w[q] = wnext[q];
    if constexpr (FRF == 4) {
        if (hm) {
            float4 v = ring_ld4(om);
            v.x += acc[0].x + prev[0].y; v.y += acc[1].x + prev[1].y; v.z += acc[2].x + prev[2].y; v.w += acc[3].x + prev[3].y;
            ring_st4(om, v);
        }
        if (hp) {
            float4 v = ring_ld4(op);
            v.x += acc[0].y + prev[0].x; v.y += acc[1].y + prev[1].x; v.z += acc[2].y + prev[2].x; v.w += acc[3].y + prev[3].x;
            ring_st4(op, v);
        }
    } else {
        static_assert(FRF == 2 || FRF == 4, "units are 2 or 4 columns wide");
        if (hm) {
            float2 v = ring_ld2(om);
            v.x += acc[0].x + prev[0].y; v.y += acc[1].x + prev[1].y;
            ring_st2(om, v);
        }
        if (hp) {
            float2 v = ring_ld2(op);
            v.x += acc[0].y + prev[0].x; v.y += acc[1].y + prev[1].x;
            ring_st2(op, v);
        }
    }
}

template <int KT, bool ADJ>
__global__ void __maxnreg__(KT <= 21 ? 160 : KT <= 25 ? 168 : (KT >= 41 && KT <= 55 && !ADJ) ? 168 : 255)
// 129 .. 168 registers leave 3 warps per scheduler.  Measured at 21 taps (cap 128 / 136 / 144 / 152 / 160 / 168: forward 0.847 / 0.767 / 0.724 /
// 0.712 / 0.696 / 0.720 ms) and at 25 (144 / 152 / 160 / 168: 1.035 / 0.951 / 0.928 / 0.915 ms): below 152 the step loop spills.  2-column units
// (41 taps and up) with 168 instead of 255: forward 41 / 51 / 55 taps 4.19 -> 3.90 / 6.09 -> 5.83 / 7.00 -> 6.56 ms per c4 arc (55 with the
// 48-column work items), adjoint slower; 63 and 75 taps spill heavily under 168.
k_conv_fold(Params P, const CpDesc *__restrict__ desc, int cp0, int n_cp, const int *__restrict__ tile_base,
            const float *__restrict__ zrad, const float *__restrict__ wtab, const float *__restrict__ in, float *__restrict__ out,
            int *item_counter, WorkCounters *wc, int in_floats, int out_floats)
{
    constexpr int C = (KT - 1) / 2;
    constexpr int FRF = fold_unit_cols(KT);           // output columns per unit
    constexpr int KP = (KT + 3) & ~3;                 // row pitch of the table image [floats]
    constexpr int WP = fold_wpitch(KT), WQ = WP / 4;  // weight row W_d[C .. 2C] in shared memory [floats], LDS.128 per row
    constexpr int XW = KT + FRF - 1;                  // window along v [columns]: 2C + FRF, even
    constexpr int NXQ = XW / 2;                       // LDS.128 per window (2 columns x 2 rows each)
    constexpr int MCX = (fold_cols_max(KT) + 2 * C + 31) / 32;       // staged columns per lane and row
    extern __shared__ float4 smem4[];
    float4 *Wd = smem4;                               // [C+1 (d)][WQ]: kernel row C+d, columns C .. 2C, zero past them
    float4 *xin4 = smem4 + (C + 1) * WQ;              // [pair][chunk]: (x[r][c], x[r+1][c], x[r][c+1], x[r+1][c+1]), chunks swizzled
    float *oring = reinterpret_cast<float *>(xin4) + in_floats;   // [slot][pitch]: ring of output rows, all zero between uses
    const unsigned xin_s = (unsigned)__cvta_generic_to_shared(xin4);
    unsigned oring_s = (unsigned)__cvta_generic_to_shared(oring);
    asm volatile("" : "+r"(oring_s));                 // an ordinary register value from here on
    const int lane = threadIdx.x;
    const int total = tile_base[n_cp];
    const int CHk = min(P.CH, C);                     // rows C+d with d > CH of an embedded smaller kernel are zero
    int slot_hint = 0;
    unsigned long long macs = 0ull;                   // multiply-adds of this lane (work counter)

    for (int e = lane; e < out_floats / 4; e += 32) reinterpret_cast<float4 *>(oring)[e] = make_float4(0.f, 0.f, 0.f, 0.f);
    __syncwarp();

    for (;;) {
        int item = 0;
        if (lane == 0) item = atomicAdd(item_counter, 1);
        item = __shfl_sync(0xffffffffu, item, 0);
        if (item >= total) break;
        while (slot_hint + 1 < n_cp && item >= tile_base[slot_hint + 1]) ++slot_hint;   // items arrive in increasing order
        const int slot = slot_hint, cp = cp0 + slot;
        const CpDesc &d = desc[cp];
        const int ncf = d.ncf, ntfc = d.ntfc, ntf = d.ntf, nts = d.nts, ri0 = d.ri0, rj0 = d.rj0, pu = d.pu, pv = d.pv;
        const int local = item - tile_base[slot];
        const int k = local / ncf, cf = local - k * ncf;
        const SliceBox S = slice_support(P, d, k);
        if (box_empty(S)) continue;
        const SliceBox F = dilate(P, S, P.CH);
        const SliceBox A = ADJ ? S : F;               // outputs to compute
        const SliceBox B = ADJ ? F : S;               // source box of the input (zero outside)
        // tiles of the chunk along v: the region's 8-column tile grid, or (one chunk) 4-column tiles from the box on
        const int ctf0 = cf * ntfc, ctf1 = min(ntf, ctf0 + ntfc);
        const int atf0 = max(ctf0, (A.v0 - rj0) / RF), atf1 = min(ctf1 - 1, (A.v1 - rj0) / RF);
        if (atf0 > atf1) continue;
        int nt = (RF / FRF) * (atf1 - atf0 + 1), av0 = rj0 + atf0 * RF;
        if (ncf == 1) {     // forward: whole 4-column (16-byte) groups from the box on, the columns k_fluence tabulates as the written box;
                            // adjoint: 8-byte aligned stores
            av0 = ADJ ? A.v0 & ~1 : A.v0 & ~3;
            nt = ADJ ? (A.v1 - av0) / FRF + 1 : (4 / FRF) * ((A.v1 - av0) / 4 + 1);
        }
        // rows: input row pairs, output rows held in the ring (T), output rows written to HBM (wu)
        const int in_u0 = B.u0, in_u1 = B.u1, npair = (in_u1 - in_u0 + 2) >> 1;
        int wu0, wu1, Tu0, Tu1;
        if (ADJ) { wu0 = Tu0 = S.u0; wu1 = Tu1 = S.u1; }
        else {      // the thread-tile rows that intersect F_k (wbox of k_fluence), clipped to the beam grid
            wu0 = ri0 + (F.u0 - ri0) / RS * RS;
            wu1 = min(P.Nu - 1, ri0 + min(nts - 1, (F.u1 - ri0) / RS) * RS + RS - 1);
            Tu0 = min(wu0, in_u0 - CHk); Tu1 = max(wu1, in_u0 + 2 * npair - 1 + CHk);
        }
        const int pitch = fold_out_pitch(nt, FRF), R = out_floats / pitch;
        const unsigned pitch_b = 4u * (unsigned)pitch, ring_bytes = pitch_b * (unsigned)R;
        const int PPc = fold_in_chunks(nt, FRF, C), maxp = fold_max_pairs(nt);
        const int ncols = FRF * nt + 2 * C;
        const long long slice_off = (long long)slot * P.stride_cp + (long long)k * pu * pv;
        const float *sbase = in + slice_off;
        float *oslice = out + slice_off + (av0 - rj0) - (long long)ri0 * pv;       // row i, column av0 + c at oslice + i pv + c

        {   // S4: columns C .. 2C of rows C .. C+CHk of the slice kernel = lerp of the table in radiological depth
            const float tz = zrad[(size_t)cp * P.Nw + k] / P.dz;
            int n0 = (int)floorf(tz);
            n0 = min(max(n0, 0), P.n_z - 2);
            const float f = fminf(fmaxf(tz - n0, 0.f), 1.f);
            const float *w0 = wtab + (size_t)n0 * KT * KP + C * KP + C, *w1 = w0 + KT * KP;
            float *Wf = reinterpret_cast<float *>(Wd);
            for (int e = lane; e < (CHk + 1) * WP; e += 32) {
                const int dd = e / WP, m = e - dd * WP;
                Wf[e] = m <= C ? (1.f - f) * __ldg(w0 + dd * KP + m) + f * __ldg(w1 + dd * KP + m) : 0.f;
            }
        }
        // flush geometry: a row has at most FOLD_COLS_MAX / 4 = 20 chunks of 16 bytes; a lane owns one chunk column and every srow-th row
        const int nchunk = (FRF * nt + 3) >> 2;
        const int srow = 32 / nchunk;
        const int lrow0 = lane / nchunk, lch0 = lane - lrow0 * nchunk;
        const int room = pv - (av0 - rj0);                 // columns of the region from av0 on
        const int fl_step = lrow0 < srow ? srow : 0x10000; // rows per trip of this lane; lanes past the last whole row sit out
        const bool col_ok = 4 * lch0 + 4 <= room, col_ok2 = 4 * lch0 + 2 <= room;
        const unsigned fl_a0 = oring_s + 16u * (unsigned)lch0, fl_a1 = fl_a0 + ring_bytes;     // the lane's chunk in ring row 0, and one ring on
        int flushed = Tu0, fslot = 0;                      // rows below `flushed` are final and written; ring slot of row `flushed`
        auto flush = [&](int b) {                          // rows [flushed, b): ring -> HBM (inside the written box), slots back to zero
            int sl = fslot + lrow0;
            while (sl >= R) sl -= R;
            unsigned ra = fl_a0 + pitch_b * (unsigned)sl;
            float *orow = oslice + (long long)(flushed + lrow0) * pv + 4 * lch0;
            for (int i = flushed + lrow0; i < b && fl_step <= 32; i += fl_step) {
                const float4 v = ring_ld4(ra);
                ring_st4(ra, make_float4(0.f, 0.f, 0.f, 0.f));
                if (i >= wu0 && i <= wu1) {
                    if (ADJ) {                             // the adjoint's columns start on an 8-byte boundary
                        if (col_ok2) *reinterpret_cast<float2 *>(orow) = make_float2(v.x, v.y);
                        if (col_ok) *reinterpret_cast<float2 *>(orow + 2) = make_float2(v.z, v.w);
                    } else if (col_ok) *reinterpret_cast<float4 *>(orow) = v;
                }
                ra += pitch_b * (unsigned)srow;
                if (ra >= fl_a1) ra -= ring_bytes;
                orow += (long long)srow * pv;
            }
            fslot += b - flushed;
            while (fslot >= R) fslot -= R;
            flushed = b;
        };

        const int n_units = npair * nt;
        // u / nt for unit indices (u < 2^16, nt < 2^8: the multiply-high by ceil(2^32 / nt) is exact)
        const unsigned nt_magic = nt > 1 ? 0xffffffffu / (unsigned)nt + 1u : 0u;
        auto div_nt = [&](int u) { return nt > 1 ? (int)__umulhi((unsigned)u, nt_magic) : u; };
        // units [u0, u1) of one group: at most 32, of at most `maxp` row pairs
        auto group_end = [&](int u0) { return min(min(n_units, u0 + 32), (div_nt(u0) + maxp) * nt); };
        // stage the input rows of a group's pairs (asynchronous copies, zero outside the source box): per-lane column terms, then one
        // pass over the rows
        auto stage = [&](int u0, int u1) {
            const int p_lo = div_nt(u0), p_hi = div_nt(u1 - 1), r_lo = in_u0 + 2 * p_lo;
            const float *sp[MCX];
            unsigned dp[MCX];
            int csz[MCX];
            bool cex[MCX];
#pragma unroll
            for (int m = 0; m < MCX; ++m) {
                const int c = lane + 32 * m, j = av0 - C + c, q = c >> 1;
                const bool cin = j >= B.v0 && j <= B.v1;
                cex[m] = c < ncols;
                csz[m] = cin ? 4 : 0;
                sp[m] = sbase + (long long)(r_lo - ri0) * pv + (cin ? j - rj0 : 0);
                dp[m] = xin_s + 16u * (unsigned)(q ^ ((q >> 3) & 1)) + 8u * (unsigned)(c & 1);
            }
            const int nrow = 2 * (p_hi - p_lo + 1);
            const int nin = min(nrow, in_u1 - r_lo + 1);          // only the second row of the last pair can lie outside the input rows
            auto rows = [&](auto ns_) {                           // ns = the column slots in use (warp-uniform)
                constexpr int ns = decltype(ns_)::value;
                unsigned ro = 0;
                for (int rl = 0; rl < nin; ++rl) {
#pragma unroll
                    for (int m = 0; m < ns; ++m) {
                        if (cex[m]) cp_async_4(dp[m] + ro, sp[m], csz[m]);
                        sp[m] += pv;
                    }
                    ro += (rl & 1) ? 16u * (unsigned)PPc - 4u : 4u;
                }
                if (nin < nrow) {
#pragma unroll
                    for (int m = 0; m < ns; ++m)
                        if (cex[m]) cp_async_4(dp[m] + ro, sbase, 0);
                }
            };
            static_assert(MCX <= 5, "column slots per lane");
            switch ((ncols + 31) >> 5) {
            case 1: rows(std::integral_constant<int, 1>{}); break;
            case 2: rows(std::integral_constant<int, MCX < 2 ? MCX : 2>{}); break;
            case 3: rows(std::integral_constant<int, MCX < 3 ? MCX : 3>{}); break;
            case 4: rows(std::integral_constant<int, MCX < 4 ? MCX : 4>{}); break;
            default: rows(std::integral_constant<int, MCX>{}); break;
            }
        };
        __syncwarp();                                      // Wd is complete; the previous item has left the ring zeroed and the staged rows free
        stage(0, group_end(0));
        for (int u0 = 0; u0 < n_units;) {
            const int u1 = group_end(u0);
            const int p_lo = div_nt(u0), p_hi = div_nt(u1 - 1);
            const int r_lo = in_u0 + 2 * p_lo, r_hi = in_u0 + 2 * p_hi;
            {   // rows that no unit from here on reaches
                const int lo = min(max(r_lo - CHk, Tu0), Tu1 + 1);
                if (lo > flushed) flush(lo);
            }
            cp_async_wait_all();
            __syncwarp();

            const int u = u0 + lane;
            const bool active = u < u1;
            const int p = active ? div_nt(u) : p_lo, t = active ? u - p * nt : 0;
            const int r = in_u0 + 2 * p;
            float2 zc[FRF], z[C][FRF];                     // folded window: zc[c] = x[j_c], z[m-1][c] = x[j_c - m] + x[j_c + m], as (row r, row r+1)
            {
                float2 xx[XW];                             // (x[r][c], x[r+1][c]) of window column c
                const float4 *xw = xin4 + (p - p_lo) * PPc;
#pragma unroll
                for (int mm = 0; mm < NXQ; ++mm) {
                    const int q = (FRF / 2) * t + mm;
                    const float4 v = xw[q ^ ((q >> 3) & 1)];
                    xx[2 * mm] = make_float2(v.x, v.y); xx[2 * mm + 1] = make_float2(v.z, v.w);
                }
                __syncwarp();                              // every lane holds its window: the staged rows are free again ...
                if (u1 < n_units) stage(u1, group_end(u1));    // ... for the next group's rows, which arrive behind this group's arithmetic
#pragma unroll
                for (int c = 0; c < FRF; ++c) {
                    zc[c] = xx[c + C];
#pragma unroll
                    for (int m = 1; m <= C; ++m) z[m - 1][c] = __fadd2_rn(xx[c + C - m], xx[c + C + m]);
                }
            }
            // steps whose two target rows lie outside the held rows for every unit of the group are skipped (adjoint halo)
            int d_lo = 0;
            if (ADJ) {
                if (r_hi + 1 < Tu0) d_lo = Tu0 - r_hi - 1;
                else if (r_lo > Tu1) d_lo = r_lo - Tu1;
            }
            if (active && CHk >= d_lo) macs += (unsigned long long)(CHk - d_lo + 1) * ((C + 1) * FRF * 2);
            int rowm = r - CHk, rowp = r + 1 + CHk;
            int sm = rowm - flushed + fslot, sp_ = rowp - flushed + fslot;     // ring slots: a few rings off at most
            while (sm < 0) sm += R;
            while (sm >= R) sm -= R;
            while (sp_ >= R) sp_ -= R;
            const float4 *wrow = Wd + CHk * WQ;
            // byte addresses of the unit's columns in its two ring rows; the "minus" row walks up the ring, the "plus" row down
            unsigned am = oring_s + 4u * (unsigned)(FRF * t + sm * pitch), ap = oring_s + 4u * (unsigned)(FRF * t + sp_ * pitch);
            const unsigned a_lo = oring_s + 4u * (unsigned)(FRF * t), a_hi = a_lo + ring_bytes;   // row 0 and one past row R - 1
            float2 accA[FRF], accB[FRF];
#pragma unroll
            for (int c = 0; c < FRF; ++c) accB[c] = make_float2(0.f, 0.f);
            float4 w[WQ];
#pragma unroll
            for (int q = 0; q < WQ; ++q) w[q] = wrow[q];
            auto held = [&](int row) { return active && (!ADJ || (row >= Tu0 && row <= Tu1)); };
            auto advance = [&]() {
                ++rowm; --rowp;
                am += pitch_b; if (am == a_hi) am = a_lo;
                if (ap == a_lo) ap = a_hi;
                ap -= pitch_b;
            };
            int dd = CHk;
#pragma unroll 1
            for (; dd > d_lo; dd -= 2) {                   // two steps per trip: the accumulators swap roles, no register copies
                fold_step<C, FRF>(zc, z, w, wrow - WQ, accA, accB, am, held(rowm), ap, held(rowp));
                advance();
                __syncwarp();                              // the rows of this step are visible to the next one
                wrow -= dd >= 2 ? 2 * WQ : WQ;             // row dd - 2 of the next trip (row 0 again after the last step: never used)
                fold_step<C, FRF>(zc, z, w, wrow, accB, accA, am, held(rowm), ap, held(rowp));
                advance();
                __syncwarp();
            }
            if (dd == d_lo) {                              // odd number of steps: the last one
                fold_step<C, FRF>(zc, z, w, wrow, accA, accB, am, held(rowm), ap, held(rowp));
                __syncwarp();
            }
            u0 = u1;
        }
        flush(Tu1 + 1);
        __syncwarp();                                      // the next item overwrites Wd and the staged rows
    }
    if (macs) atomicAdd(reinterpret_cast<unsigned long long *>(ADJ ? &wc->macs_adj : &wc->macs_fwd), macs);
}

}  // namespace pdrt
