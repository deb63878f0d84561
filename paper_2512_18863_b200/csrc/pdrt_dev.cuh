// pdrt_dev.cuh — device-side parameter blocks and geometry helpers shared by all kernels.
//
// Data layout in HBM:
//   density, dose, dL/dDose : patient grid [nz][ny][nx] float32
//   phimap, gphimap, P0, ... : [n_cp][Nvf][Nuf] float32, valid only inside the fluence support
//                              bbox of each control point (CpDesc a0..a1, b0..b1)
//   zrad                    : [n_cp][Nw] float32
//   phimapT                 : [n_cp][Nuf][Nvf] float32, the same maps with v fastest (read by the conv tile fill)
//   gT                      : dL/dDose transposed to [ny][nx][nz] (z fastest)
//   D_b / H_b               : per control point a COMPACT beam-frame block, layout [w][u][v], v FASTEST:
//        index(cp; i,j,k) = cp_slot*stride_cp + (k*pu + (i - ri0))*pv + (j - rj0)
//     covering the region [ri0, ri0+pu) x [rj0, rj0+pv) x [0, Nw) that bounds the conv footprint
//     of that control point (jaw opening magnified per slice, dilated by blur and kernel halo);
//     rj0 % 8 == 0, pv % 8 == 0, pu % RS == 0, rows / columns past the beam grid hold zeros.
//     The gantry rotates about patient z = beam v (G1), so the bilinear weights of the
//     beam <-> patient resampling do not depend on v: with v fastest every resampling thread computes
//     its weights once and then streams 16-byte vectors along v.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace pdrt {

constexpr int RF = 8;              // conv outputs per thread along v (the fast, register-window axis)
constexpr int RS = 2;              // conv outputs per thread along u (the slow axis)
constexpr int CONV_THREADS = 32;   // the conv runs one warp per block (no block-level barriers)
constexpr int NTFC_MAX = 8;        // conv chunk width in thread-tiles along v (64 outputs)
constexpr int CONV_CHUNK_TILES = 32;  // thread-tiles per conv chunk: one per lane
constexpr int MAX_TAPS = 64;       // largest Gaussian half-width [pixels]
constexpr int MAX_HS = 4;          // largest number of head-scatter Gaussians

struct Params {
    // patient grid
    int nx, ny, nz;
    float sx, sy, sz, ox, oy, oz, isox, isoy, isoz;
    // beam grid (Nv = nz, dv = sz)
    int Nu, Nv, Nw;
    float du, dv, dw, wmin, cu, v0;      // cu = (Nu-1)/2, v0 = oz - iso_z  (v_j = v0 + j dv)
    // fluence map
    int Nuf, Nvf;
    float Du, Dv, cuf, cvf;              // cuf = (Nuf-1)/2
    float sid, tau, cal;
    int Np;                              // leaf pairs
    // lateral kernel
    int K, KT;                           // requested size; compiled variant of ONE pass (single pass: KT >= K)
    int NB, CH;                          // passes per axis (odd): the K x K kernel, centred in an (NB KT)^2 window, is applied as NB^2
                                         // KT x KT sub-kernels with shifted inputs;  CH = (K-1)/2, the halo of the footprint F_k
    int n_z;
    float dz;
    int tile_floats;                     // conv input-tile budget in shared memory [floats]
    int ntfc_max;                        // widest conv work item [thread-tiles along v]: NTFC_MAX (k_conv) or SYM_NTFC_MAX (k_conv_sym)
    int conv_sym;                        // 0: k_conv; 1: k_conv_sym (row-symmetric); 2: k_conv_fold (row- and column-symmetric); the last two count their own multiply-adds
    // fluence corrections
    int Tu_max, Tv_max;                  // largest Gaussian half-widths along u / v
    // ray marcher
    int M_ray;
    double ray_step;
    // compact beam-frame blocks
    long long stride_cp;                 // floats per control point
};

// Gaussian taps and tables of the fluence corrections (device pointers into one float pool).
struct FluTables {
    const float *leaf_bounds;            // [Np+1]
    const float *oar;                    // [n_oar]
    int n_oar;
    float oar_dr;
    int Tu, Tv;                          // penumbra half-widths: MLC (along u), jaw (along v)
    const float *gu, *gv;                // [2Tu+1], [2Tv+1]
    int n_hs;
    float hs_amp[MAX_HS];
    int hs_Tu[MAX_HS], hs_Tv[MAX_HS];
    const float *hs_gu[MAX_HS], *hs_gv[MAX_HS];
};

// Per-control-point descriptor, built on the device by k_fluence (no host sync on the path).
struct CpDesc {
    float cg, sg;                // cos / sin of the gantry angle
    float scale;                 // cal * MU
    int a0, a1, b0, b1;          // fluence support bbox in the COLLIMATOR frame (inclusive); empty when a0 > a1
    int pa0, pa1, pb0, pb1;      // the same in the PROJECTION frame (after the collimator rotation; equal to a0.. when the angle is 0):
                                 // what S3 / S9 and every slice box are derived from
    float cc, sc;                // cos / sin of the collimator angle
    int ja0, ja1, jb0, jb1;      // jaw bbox (pixels where Phi0 or its jaw derivative can be non-zero)
    int ri0, rj0, pu, pv;        // compact region origin and extents (rj0 % 8 == 0, pv % 8 == 0, pu % RS == 0)
    int ntf, nts;                // region size in thread-tiles: RF along v (fast), RS along u (slow)
    int ncf, ntfc;               // conv chunks along v and their width [thread-tiles]
    int n_items, n_items_adj;    // Nw * ncf conv work items, forward / adjoint (0 when empty)
    unsigned long long support_vox, footprint_vox, region_vox, macs_fwd, macs_adj;
};

struct WorkCounters {
    long long items, support_vox, footprint_vox, region_vox, macs_fwd, macs_adj, fan_rays;
};

// Row pitch [floats] of the conv input tile for `naf` thread-tiles along v: the (K+7)-wide register window of
// the last thread-tile must fit, rounded to 8 floats so that the quad swizzle stays inside the row.
__host__ __device__ __forceinline__ int conv_pitch(int kt, int naf)
{
    const int xw = (kt + RF - 1 + 3) & ~3;
    return (naf * RF + xw - RF + 7) & ~7;
}

struct SliceBox { int u0, u1, v0, v1; };   // inclusive voxel-index box; empty when u0 > u1 or v0 > v1

// Per (control point, slice) boxes tabulated once per call by k_fluence ([n_cp][Nw], 8 bytes each, L2-resident), so that
// the resampling kernels read a box instead of re-deriving it per beam row / patient column:
//   sbox = S_k;  wbox = the part of slice k of D_b that the forward conv writes (F_k rounded outward to thread-tiles,
//   clipped to the beam grid) — outside it the compact block holds stale data and must not be read.
struct __align__(8) SliceBox16 { short u0, u1, v0, v1; };
__device__ __forceinline__ SliceBox16 load_box(const SliceBox16 *__restrict__ t, size_t idx)
{
    const int2 r = __ldg(reinterpret_cast<const int2 *>(t) + idx);
    SliceBox16 b;
    b.u0 = (short)(r.x & 0xffff); b.u1 = (short)(r.x >> 16); b.v0 = (short)(r.y & 0xffff); b.v1 = (short)(r.y >> 16);
    return b;
}

__device__ __forceinline__ bool box_empty(const SliceBox &b) { return b.u0 > b.u1 || b.v0 > b.v1; }

// S_k: beam voxels of slice k whose bilinear stencil (Eq. 5) can touch a pixel of the fluence
// support bbox (projection frame), i.e. fa in (pa0-1, pa1+1), fb in (pb0-1, pb1+1); rounded outward, clipped to the grid.
// Every kernel derives its per-slice extents from this one function.
__device__ __forceinline__ SliceBox slice_support(const Params &P, const CpDesc &d, int k)
{
    const float inv_mag = (P.sid + P.wmin + k * P.dw) / P.sid;
    const float ulo = (d.pa0 - 1 - P.cuf) * P.Du * inv_mag, uhi = (d.pa1 + 1 - P.cuf) * P.Du * inv_mag;
    const float vlo = (d.pb0 - 1 - P.cvf) * P.Dv * inv_mag, vhi = (d.pb1 + 1 - P.cvf) * P.Dv * inv_mag;
    SliceBox s;
    s.u0 = max(0, (int)floorf(ulo / P.du + P.cu));
    s.u1 = min(P.Nu - 1, (int)ceilf(uhi / P.du + P.cu));
    s.v0 = max(0, (int)floorf((vlo - P.v0) / P.dv));
    s.v1 = min(P.Nv - 1, (int)ceilf((vhi - P.v0) / P.dv));
    return s;
}

// F_k = S_k dilated by the kernel half-width, clipped to the beam grid.
__device__ __forceinline__ SliceBox dilate(const Params &P, const SliceBox &s, int c)
{
    SliceBox f;
    f.u0 = max(0, s.u0 - c); f.u1 = min(P.Nu - 1, s.u1 + c);
    f.v0 = max(0, s.v0 - c); f.v1 = min(P.Nv - 1, s.v1 + c);
    if (box_empty(s)) { f.u0 = 1; f.u1 = 0; }
    return f;
}

__device__ __forceinline__ size_t compact_index(const Params &P, const CpDesc &d, int slot, int i, int j, int k)
{
    return (size_t)slot * (size_t)P.stride_cp + ((size_t)k * d.pu + (i - d.ri0)) * d.pv + (j - d.rj0);
}

// Eq. 4: fractional overlap of [lo,hi] with the pixel centred at c, width D.
__device__ __forceinline__ float ov(float c, float D, float lo, float hi)
{
    const float a = fminf(hi, c + 0.5f * D) - fmaxf(lo, c - 0.5f * D);
    return a > 0.f ? a / D : 0.f;
}
// Subgradients of Eq. 4 with the half-open convention of DESIGN.md G9.
__device__ __forceinline__ float dov_dhi(float c, float D, float lo, float hi)
{
    const float pl = c - 0.5f * D, pr = c + 0.5f * D;
    return (pl <= hi && hi < pr && hi >= fmaxf(lo, pl)) ? 1.f / D : 0.f;
}
__device__ __forceinline__ float dov_dlo(float c, float D, float lo, float hi)
{
    const float pl = c - 0.5f * D, pr = c + 0.5f * D;
    return (pl < lo && lo <= pr && lo <= fminf(hi, pr)) ? -1.f / D : 0.f;
}

__device__ __forceinline__ float warp_sum(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

}  // namespace pdrt
