// pdrt_conv_sym.cuh — S4+S5 (forward) and S8 (adjoint): the per-slice lateral convolution (Eq. 8) in
// ROW-SYMMETRIC form (runs at 11 taps; pdrt_conv_fold.cuh adds the column symmetry and serves 15-75 taps).
//
// The pencil kernel is radially symmetric and its pixel-integrated table is built mirrored (R3), so
// W[C+d][.] = W[C-d][.].  With the row correlation
//     T_d[r][j] = sum_dj W[C+d][dj] x[r][j + dj - C],        d = 0 .. C,
// every output row is  out[i] = T_0[i] + sum_{d=1..C} (T_d[i+d] + T_d[i-d]):  a row correlation of INPUT row r is computed
// once and added to the TWO output rows r-d and r+d.  That is (C+1) KT multiply-adds per input value instead of KT^2, and
// the loop runs over the rows that hold input (S_k forward: no multiply-adds on the structurally zero rows of the halo;
// F_k adjoint), not over output rows.
//
// One WARP per block, persistent over the work items (control point, slice, chunk along v) like k_conv.  A lane owns a UNIT =
// (pair of input rows r, r+1) x (8 output columns): the (KT+7)-wide window of both rows sits in registers as float2 (row r,
// row r+1), the weights come as warp-broadcast LDS.128 (four taps each; FFMA2 takes a tap as a scalar operand for both halves),
// and one packed FFMA2 per tap and column yields (a_d, b_d) = (T_d[r], T_d[r+1]).  Output rows are accumulated in a
// shared-memory RING of rows private to the warp; since out[r-d] takes a_d + b_{d+1} and out[r+1+d] takes b_d + a_{d+1},
// walking d downwards with the previous (a, b) kept in registers costs ONE read-modify-write of 8 columns per side and step.  In one step the "minus" rows r-d (parity of d) and
// the "plus" rows r+1+d (other parity) cannot coincide, and the lanes of a group hold distinct (row pair, tile), so a step
// has no write conflicts; one __syncwarp per step orders the steps.  Rows that no later unit can reach are written to HBM
// and their ring slots zeroed.  The input rows of the 32 units in flight are staged with cp.async (zero-filled outside the
// source box), interleaved by row pair so that a window load is LDS.128.
#pragma once
#include "pdrt_conv.cuh"

namespace pdrt {

constexpr int SYM_NTFC_MAX = 10;       // widest work item [thread-tiles of 8 columns along v]

// Ring row [floats]: columns 0-3 of every tile first, then columns 4-7 (second plane at 4 nt), so that the two LDS.128 of a
// read-modify-write hit consecutive 16-byte chunks across the lanes of a row.  The lanes of a quarter-warp that fall on the
// next row pair are two rows on: the pitch is padded until that offset (pitch/2 chunks, modulo the 8 chunks of a wavefront)
// continues where the row ends, give or take one chunk.
__host__ __device__ __forceinline__ int sym_out_pitch(int nt)
{
    int p = 8 * nt;
    for (;; p += 4) {
        const int dl = (p >> 1) & 7;
        if (dl == (nt & 7) || dl == ((nt + 1) & 7) || dl == ((nt - 1) & 7)) return p;
    }
}
// row pairs per group of units: as many whole-or-part pairs as 32 units span, at most 8
__host__ __device__ __forceinline__ int sym_max_pairs(int nt) { return (32 + nt - 1) / nt < 8 ? (32 + nt - 1) / nt : 8; }
// 16-byte chunks (2 columns x 2 rows) per staged row pair: the windows of nt tiles, rounded to the 8-chunk swizzle period
__host__ __device__ __forceinline__ int sym_in_chunks(int nt, int c) { return (4 * nt + c + 7) & ~7; }
inline int sym_out_floats(int kt)
{
    const int c = (kt - 1) / 2;
    int best = 0;
    for (int nt = 1; nt <= SYM_NTFC_MAX; ++nt) best = std::max(best, (2 * sym_max_pairs(nt) + 2 * c) * sym_out_pitch(nt));
    return best;
}
inline int sym_in_floats(int kt)
{
    const int c = (kt - 1) / 2;
    int best = 0;
    for (int nt = 1; nt <= SYM_NTFC_MAX; ++nt) best = std::max(best, sym_max_pairs(nt) * sym_in_chunks(nt, c) * 4);
    return best;
}
inline size_t sym_smem_bytes(int kt)
{
    const int c = (kt - 1) / 2, kp = (kt + 3) & ~3;
    return sizeof(float) * ((size_t)(c + 1) * kp + sym_in_floats(kt) + sym_out_floats(kt));
}

__device__ __forceinline__ int pmod(int a, int m) { const int r = a % m; return r < 0 ? r + m : r; }

// One step d of a unit: acc = (a_d, b_d) from the window and the weight row `w` (registers); then the weight row of the NEXT step is
// fetched into `w` (its latency hides behind the read-modify-writes) and out[r-d] += a_d + b_{d+1}, out[r+1+d] += b_d + a_{d+1},
// with (a_{d+1}, b_{d+1}) = prev.  `om` / `op` point at the unit's 8 columns (first plane) of the two ring rows; null: row not held.
template <int KT>
__device__ __forceinline__ void sym_step(const float2 (&xx)[KT + 7], float4 (&w)[(KT + 3) / 4], const float4 *__restrict__ wnext,
                                         float2 (&acc)[RF], const float2 (&prev)[RF], float *om, float *op, int hp)
{
    constexpr int KQ4 = (KT + 3) / 4;
#pragma unroll
    for (int q = 0; q < KQ4; ++q) {
        const float ws[4] = { w[q].x, w[q].y, w[q].z, w[q].w };
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int dj = 4 * q + e;
            if (dj < KT) {
                const float2 wd = make_float2(ws[e], ws[e]);          // one register: FFMA2 takes it as a scalar operand
#pragma unroll
                for (int c = 0; c < RF; ++c) acc[c] = dj == 0 ? __fmul2_rn(xx[c], wd) : __ffma2_rn(xx[c + dj], wd, acc[c]);
            }
        }
    }
#pragma unroll
    for (int q = 0; q < KQ4; ++q) w[q] = wnext[q];
    if (om) {
        float4 *o = reinterpret_cast<float4 *>(om), *o2 = reinterpret_cast<float4 *>(om + hp);
        float4 v0 = *o, v1 = *o2;
        v0.x += acc[0].x + prev[0].y; v0.y += acc[1].x + prev[1].y; v0.z += acc[2].x + prev[2].y; v0.w += acc[3].x + prev[3].y;
        v1.x += acc[4].x + prev[4].y; v1.y += acc[5].x + prev[5].y; v1.z += acc[6].x + prev[6].y; v1.w += acc[7].x + prev[7].y;
        *o = v0; *o2 = v1;
    }
    if (op) {
        float4 *o = reinterpret_cast<float4 *>(op), *o2 = reinterpret_cast<float4 *>(op + hp);
        float4 v0 = *o, v1 = *o2;
        v0.x += acc[0].y + prev[0].x; v0.y += acc[1].y + prev[1].x; v0.z += acc[2].y + prev[2].x; v0.w += acc[3].y + prev[3].x;
        v1.x += acc[4].y + prev[4].x; v1.y += acc[5].y + prev[5].x; v1.z += acc[6].y + prev[6].x; v1.w += acc[7].y + prev[7].x;
        *o = v0; *o2 = v1;
    }
}

// resident warps per SM the register allocation aims at (the window takes 2 (KT + 7) registers)
constexpr int sym_min_blocks(int kt) { return kt <= 25 ? 14 : kt <= 31 ? 11 : 8; }

template <int KT, bool ADJ>
__global__ void __launch_bounds__(CONV_THREADS, sym_min_blocks(KT))
k_conv_sym(Params P, const CpDesc *__restrict__ desc, int cp0, int n_cp, const int *__restrict__ tile_base,
           const float *__restrict__ zrad, const float *__restrict__ wtab, const float *__restrict__ in, float *__restrict__ out,
           int *item_counter, WorkCounters *wc, int in_floats, int out_floats)
{
    constexpr int C = (KT - 1) / 2;
    constexpr int KP = (KT + 3) & ~3;                 // row pitch of the table image and of Wd [floats]
    constexpr int KQ4 = KP / 4;                       // LDS.128 per weight row
    constexpr int XW = KT + 7;                        // register window along v [columns], even
    constexpr int NXQ = XW / 2;                       // LDS.128 per window (2 columns x 2 rows each)
    constexpr int MCX = (8 * SYM_NTFC_MAX + 2 * C + 31) / 32;    // staged columns per lane and row
    extern __shared__ float4 smem4[];
    float4 *Wd = smem4;                               // [C+1 (d)][KQ4]: kernel row C+d, zero past KT
    float4 *xin4 = smem4 + (C + 1) * KQ4;             // [pair][chunk]: (x[r][c], x[r+1][c], x[r][c+1], x[r+1][c+1]), chunks swizzled
    float *oring = reinterpret_cast<float *>(xin4) + in_floats;   // [slot][pitch]: ring of output rows, all zero between uses
    const unsigned xin_s = (unsigned)__cvta_generic_to_shared(xin4);
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
        // tiles of the chunk along v
        const int ctf0 = cf * ntfc, ctf1 = min(ntf, ctf0 + ntfc);
        const int atf0 = max(ctf0, (A.v0 - rj0) / RF), atf1 = min(ctf1 - 1, (A.v1 - rj0) / RF);
        if (atf0 > atf1) continue;
        int nt = atf1 - atf0 + 1, av0 = rj0 + atf0 * RF;
        if (ncf == 1) {     // one chunk: the tiles start at the box instead of the region's tile grid (fewer tiles; k_fluence tabulates the same
                            // columns as the written box); forward stores are 16-byte, adjoint stores 8-byte aligned
            av0 = ADJ ? A.v0 & ~1 : A.v0 & ~3;
            nt = (A.v1 - av0) / RF + 1;
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
        const int pitch = sym_out_pitch(nt), hp = 4 * nt, R = out_floats / pitch;
        const int PPc = sym_in_chunks(nt, C), maxp = sym_max_pairs(nt);
        const int ncols = 8 * nt + 2 * C;
        const long long slice_off = (long long)slot * P.stride_cp + (long long)k * pu * pv;
        const float *sbase = in + slice_off;
        float *oslice = out + slice_off + (av0 - rj0) - (long long)ri0 * pv;       // row i, column av0 + c at oslice + i pv + c

        {   // S4: rows C .. C+CHk of the slice kernel = lerp of the table in radiological depth
            const float tz = zrad[(size_t)cp * P.Nw + k] / P.dz;
            int n0 = (int)floorf(tz);
            n0 = min(max(n0, 0), P.n_z - 2);
            const float f = fminf(fmaxf(tz - n0, 0.f), 1.f);
            const float4 *w0 = reinterpret_cast<const float4 *>(wtab + (size_t)n0 * KT * KP + C * KP), *w1 = w0 + KT * KQ4;
            for (int e = lane; e < (CHk + 1) * KQ4; e += 32) {
                const float4 a = __ldg(w0 + e), b = __ldg(w1 + e);
                Wd[e] = make_float4((1.f - f) * a.x + f * b.x, (1.f - f) * a.y + f * b.y, (1.f - f) * a.z + f * b.z, (1.f - f) * a.w + f * b.w);
            }
        }
        // flush geometry: the lanes walk the 16-byte (forward) / 8-byte (adjoint) chunks of consecutive rows, 32 chunks per trip
        const int nchunk = ADJ ? 4 * nt : 2 * nt;
        const int lrow0 = lane / nchunk, lch0 = lane - lrow0 * nchunk, srow = 32 / nchunk, sch = 32 - srow * nchunk;
        const int room = pv - (av0 - rj0);                 // columns of the region from av0 on
        int flushed = Tu0, fslot = 0;                      // rows below `flushed` are final and written; ring slot of row `flushed`
        auto flush = [&](int b) {                          // rows [flushed, b): ring -> HBM (inside the written box), slots back to zero
            int i = flushed + lrow0, ch = lch0, sl = fslot + lrow0;
            while (sl >= R) sl -= R;
            while (__any_sync(0xffffffffu, i < b)) {
                if (i < b) {
                    float *rowp = oring + sl * pitch;
                    const bool wr = i >= wu0 && i <= wu1;
                    float *orow = oslice + (long long)i * pv;
                    if (ADJ) {
                        const int c = 2 * ch;
                        float2 *p = reinterpret_cast<float2 *>(rowp + ((c >> 2) & 1) * hp + 4 * (c >> 3) + (c & 3));
                        const float2 v = *p;
                        *p = make_float2(0.f, 0.f);
                        if (wr && c + 2 <= room) *reinterpret_cast<float2 *>(orow + c) = v;
                    } else {
                        float4 *p = reinterpret_cast<float4 *>(rowp + (ch & 1) * hp + 4 * (ch >> 1));
                        const float4 v = *p;
                        *p = make_float4(0.f, 0.f, 0.f, 0.f);
                        if (wr && 4 * ch + 4 <= room) *reinterpret_cast<float4 *>(orow + 4 * ch) = v;
                    }
                }
                ch += sch; i += srow; sl += srow;
                if (ch >= nchunk) { ch -= nchunk; ++i; ++sl; }
                while (sl >= R) sl -= R;
            }
            fslot += b - flushed;
            while (fslot >= R) fslot -= R;
            flushed = b;
        };

        const int n_units = npair * nt;
        __syncwarp();                                      // Wd is complete; the previous item has left the ring zeroed
        for (int u0 = 0; u0 < n_units;) {
            const int p_lo = u0 / nt;
            const int u1 = min(min(n_units, u0 + 32), (p_lo + maxp) * nt);       // units [u0, u1) of at most `maxp` row pairs
            const int p_hi = (u1 - 1) / nt;
            const int r_lo = in_u0 + 2 * p_lo, r_hi = in_u0 + 2 * p_hi;
            {   // rows that no unit from here on reaches
                const int lo = min(max(r_lo - CHk, Tu0), Tu1 + 1);
                if (lo > flushed) flush(lo);
            }
            {   // stage the input rows of the group's pairs: per-lane column terms, then one pass over the rows
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
                    dp[m] = xin_s + 16u * (unsigned)(q ^ ((q >> 3) & 7)) + 8u * (unsigned)(c & 1);
                }
                const int nrow = 2 * (p_hi - p_lo + 1);
                const int nin = min(nrow, in_u1 - r_lo + 1);      // only the second row of the last pair can lie outside the input rows
                unsigned ro = 0;
                for (int rl = 0; rl < nin; ++rl) {
#pragma unroll
                    for (int m = 0; m < MCX; ++m) {
                        if (cex[m]) cp_async_4(dp[m] + ro, sp[m], csz[m]);
                        sp[m] += pv;
                    }
                    ro += (rl & 1) ? 16u * (unsigned)PPc - 4u : 4u;
                }
                if (nin < nrow) {
#pragma unroll
                    for (int m = 0; m < MCX; ++m)
                        if (cex[m]) cp_async_4(dp[m] + ro, sbase, 0);
                }
            }
            cp_async_wait_all();
            __syncwarp();

            const int u = u0 + lane;
            const bool active = u < u1;
            const int p = active ? u / nt : p_lo, t = active ? u - p * nt : 0;
            const int r = in_u0 + 2 * p;
            float2 xx[XW];                                 // (x[r][c], x[r+1][c]) of window column c
            {
                const float4 *xw = xin4 + (p - p_lo) * PPc;
#pragma unroll
                for (int mm = 0; mm < NXQ; ++mm) {
                    const int q = 4 * t + mm;
                    const float4 v = xw[q ^ ((q >> 3) & 7)];
                    xx[2 * mm] = make_float2(v.x, v.y); xx[2 * mm + 1] = make_float2(v.z, v.w);
                }
            }
            // steps whose two target rows lie outside the held rows for every unit of the group are skipped (adjoint halo)
            int d_lo = 0;
            if (ADJ) {
                if (r_hi + 1 < Tu0) d_lo = Tu0 - r_hi - 1;
                else if (r_lo > Tu1) d_lo = r_lo - Tu1;
            }
            if (active && CHk >= d_lo) macs += (unsigned long long)(CHk - d_lo + 1) * (KT * RF * 2);
            // ring rows of the two sides: r - d walks up the ring as d falls, r + 1 + d walks down; an inactive lane or a row
            // that is not held gets no address
            int rowm = r - CHk, rowp = r + 1 + CHk;
            int sm = pmod(rowm - flushed + fslot, R), sp_ = pmod(rowp - flushed + fslot, R);
            const float4 *wrow = Wd + CHk * KQ4;
            float *const obase = oring + 4 * t;
            float2 accA[RF], accB[RF];
#pragma unroll
            for (int c = 0; c < RF; ++c) accB[c] = make_float2(0.f, 0.f);
            float4 w[KQ4];
#pragma unroll
            for (int q = 0; q < KQ4; ++q) w[q] = wrow[q];
            auto held = [&](int row) { return active && (!ADJ || (row >= Tu0 && row <= Tu1)); };
            int dd = CHk;
#pragma unroll 1
            for (; dd > d_lo; dd -= 2) {                   // two steps per trip: the accumulators swap roles, no register copies
                sym_step<KT>(xx, w, wrow - KQ4, accA, accB, held(rowm) ? obase + sm * pitch : nullptr, held(rowp) ? obase + sp_ * pitch : nullptr, hp);
                ++rowm; --rowp; sm = sm + 1 == R ? 0 : sm + 1; sp_ = sp_ == 0 ? R - 1 : sp_ - 1;
                __syncwarp();                              // the rows of this step are visible to the next one
                wrow -= dd >= 2 ? 2 * KQ4 : KQ4;           // row dd - 2 of the next trip (row 0 again after the last step: never used)
                sym_step<KT>(xx, w, wrow, accB, accA, held(rowm) ? obase + sm * pitch : nullptr, held(rowp) ? obase + sp_ * pitch : nullptr, hp);
                ++rowm; --rowp; sm = sm + 1 == R ? 0 : sm + 1; sp_ = sp_ == 0 ? R - 1 : sp_ - 1;
                __syncwarp();
            }
            if (dd == d_lo) {                              // odd number of steps: the last one
                sym_step<KT>(xx, w, wrow, accA, accB, held(rowm) ? obase + sm * pitch : nullptr, held(rowp) ? obase + sp_ * pitch : nullptr, hp);
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
