// pdrt_depth.cuh — S2 radiological depth (Eq. 7): one central-axis ray per gantry
// angle, uniform midpoint samples from the source, trilinear density lookup, prefix sum, and the
// depth of every beam-grid slice by linear interpolation of the running sum (G7, G8).
// Positions, the in-box decision and the prefix sum are float64 so that the sample that straddles
// the grid face is classified exactly as a float64 reference would (it decides a whole step of depth).
#pragma once
#include "pdrt_dev.cuh"

namespace pdrt {

constexpr int DEPTH_THREADS = 256;

__device__ __forceinline__ double density_at(const Params &P, const float *__restrict__ rho, double px, double py, double pz)
{
    const double p[3] = { px, py, pz };
    const double o[3] = { (double)P.ox, (double)P.oy, (double)P.oz }, s[3] = { (double)P.sx, (double)P.sy, (double)P.sz };
    const int N[3] = { P.nx, P.ny, P.nz };
    int i0[3], i1[3];
    double t[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (p[a] < o[a] - 0.5 * s[a] || p[a] > o[a] + (N[a] - 0.5) * s[a]) return 0.0;
        const double f = (p[a] - o[a]) / s[a];
        const int fl = (int)floor(f);
        t[a] = f - fl;
        i0[a] = min(max(fl, 0), N[a] - 1);
        i1[a] = min(max(fl + 1, 0), N[a] - 1);
    }
    double acc = 0.0;
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const int ix = (c & 1) ? i1[0] : i0[0], iy = (c & 2) ? i1[1] : i0[1], iz = (c & 4) ? i1[2] : i0[2];
        const double wx = (c & 1) ? t[0] : 1.0 - t[0], wy = (c & 2) ? t[1] : 1.0 - t[1], wz = (c & 4) ? t[2] : 1.0 - t[2];
        acc += wx * wy * wz * (double)__ldg(&rho[((size_t)iz * P.ny + iy) * P.nx + ix]);
    }
    return acc;
}

// The same lookup for the ray bundle of the divergent-depth mode: position, in-box decision and cell index in float64 (the
// decision a float64 reference takes), interpolation weights and arithmetic in float32.
__device__ __forceinline__ float density_at_f(const Params &P, const float *__restrict__ rho, const double (&inv_s)[3], double px, double py, double pz)
{
    const double p[3] = { px, py, pz };
    const double o[3] = { (double)P.ox, (double)P.oy, (double)P.oz }, s[3] = { (double)P.sx, (double)P.sy, (double)P.sz };
    const int N[3] = { P.nx, P.ny, P.nz };
    int i0[3], i1[3];
    float t[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (p[a] < o[a] - 0.5 * s[a] || p[a] > o[a] + (N[a] - 0.5) * s[a]) return 0.f;     // the box decision: in float64, as a reference takes it
        const double f = (p[a] - o[a]) * inv_s[a];                                          // the cell index may differ by rounding only on a cell
        const double fl = floor(f);                                                         // boundary, where the interpolant is continuous
        t[a] = (float)(f - fl);
        i0[a] = min(max((int)fl, 0), N[a] - 1);
        i1[a] = min(max((int)fl + 1, 0), N[a] - 1);
    }
    const float *r00 = rho + ((size_t)i0[2] * P.ny + i0[1]) * P.nx, *r01 = rho + ((size_t)i0[2] * P.ny + i1[1]) * P.nx;
    const float *r10 = rho + ((size_t)i1[2] * P.ny + i0[1]) * P.nx, *r11 = rho + ((size_t)i1[2] * P.ny + i1[1]) * P.nx;
    const float a00 = __ldg(r00 + i0[0]) + t[0] * (__ldg(r00 + i1[0]) - __ldg(r00 + i0[0]));
    const float a01 = __ldg(r01 + i0[0]) + t[0] * (__ldg(r01 + i1[0]) - __ldg(r01 + i0[0]));
    const float a10 = __ldg(r10 + i0[0]) + t[0] * (__ldg(r10 + i1[0]) - __ldg(r10 + i0[0]));
    const float a11 = __ldg(r11 + i0[0]) + t[0] * (__ldg(r11 + i1[0]) - __ldg(r11 + i0[0]));
    const float b0 = a00 + t[1] * (a01 - a00), b1 = a10 + t[1] * (a11 - a10);
    return b0 + t[2] * (b1 - b0);
}

// Grid: n_cp blocks.  rho_s [n_cp][M], Z_s [n_cp][M+1] are float64 scratch; zrad [n_cp][Nw] float32.
__global__ void __launch_bounds__(DEPTH_THREADS)
k_depth(Params P, int n_cp, const float *__restrict__ rho, const float *__restrict__ gantry_deg,
        double *rho_s, double *Z_s, float *zrad)
{
    const int cp = blockIdx.x, tid = threadIdx.x;
    if (cp >= n_cp) return;
    const int M = P.M_ray;
    double *r = rho_s + (size_t)cp * M, *Z = Z_s + (size_t)cp * (M + 1);
    const double phi = (double)gantry_deg[cp] * 3.14159265358979323846 / 180.0;
    const double wx = -sin(phi), wy = cos(phi);
    const double srcx = (double)P.isox - (double)P.sid * wx, srcy = (double)P.isoy - (double)P.sid * wy, srcz = (double)P.isoz;
    const double ds = P.ray_step;
    // each thread owns a contiguous run of samples
    const int per = (M + DEPTH_THREADS - 1) / DEPTH_THREADS;
    const int m_lo = min(M, tid * per), m_hi = min(M, m_lo + per);
    double run = 0.0;
    for (int m = m_lo; m < m_hi; ++m) {
        const double t = (m + 0.5) * ds;
        const double v = density_at(P, rho, srcx + t * wx, srcy + t * wy, srcz);
        r[m] = v;
        run += v * ds;
    }
    // exclusive scan of the per-thread sums: shuffle scan inside each warp, then the warp totals in warp order (fixed order of additions)
    __shared__ double wtot[DEPTH_THREADS / 32];
    double incl = run;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const double up = __shfl_up_sync(0xffffffffu, incl, o);
        if ((tid & 31) >= o) incl += up;
    }
    if ((tid & 31) == 31) wtot[tid >> 5] = incl;
    __syncthreads();
    double z = incl - run;
    for (int w = 0; w < (tid >> 5); ++w) z += wtot[w];
    for (int m = m_lo; m < m_hi; ++m) { Z[m] = z; z += r[m] * ds; }
    if (m_hi == M && m_lo < M) Z[M] = z;
    if (M == 0 && tid == 0) Z[0] = 0.0;
    __syncthreads();
    for (int k = tid; k < P.Nw; k += DEPTH_THREADS) {
        const double q = ((double)P.sid + (double)P.wmin + k * (double)P.dw) / ds;
        float out = 0.f;
        if (q > 0.0) {
            const int m0 = min((int)floor(q), M - 1);
            out = (float)(Z[m0] + (q - m0) * r[m0] * ds);
        }
        zrad[(size_t)cp * P.Nw + k] = out;
    }
}

// ---------------------------------------------------------------------------------------------------------------
// Divergent radiological depth (optional mode; reading G24 of DESIGN.md).  One diverging ray per
// fluence-map pixel (a,b) of the support bbox (grown by one pixel, for the interpolation): from the source through
// (uf_a, vf_b) on the isocentre plane, P(t) = source + t (w^ + uf/SID u^ + vf/SID v^), t = distance along the axis; Eq. 7
// with the sampling rule of the central-axis ray in t, so depth counts per unit axial distance and a medium that is
// homogeneous across the beam gives every ray the central-axis profile.  At every slice the depth factor
//   F[k][b][a] = T(z_fan) / T(z_cax[k])   (1 where T(z_cax[k]) <= 0),   T(z) = 2 pi (A/a + B/b)(z)  (plane integral of K)
// is stored; k_apply_fan multiplies the projected fluence (forward) resp. H_b (adjoint) by its bilinear interpolant.
struct FanBox { int a0, b0, bw, bh; };     // pixels [a0, a0+bw) x [b0, b0+bh) of the control point's rays
__device__ __forceinline__ FanBox fan_box(const Params &P, const CpDesc &d)
{
    FanBox f;
    f.a0 = max(0, d.pa0 - 1); f.b0 = max(0, d.pb0 - 1);
    f.bw = min(P.Nuf - 1, d.pa1 + 1) - f.a0 + 1; f.bh = min(P.Nvf - 1, d.pb1 + 1) - f.b0 + 1;
    return f;
}
__device__ __forceinline__ float depth_term(const float *__restrict__ Ttab, int n_z, float dz, float z)
{
    const float t = z / dz;
    int n0 = (int)floorf(t);
    n0 = min(max(n0, 0), n_z - 2);
    const float f = fminf(fmaxf(t - n0, 0.f), 1.f);
    return (1.f - f) * __ldg(Ttab + n0) + f * __ldg(Ttab + n0 + 1);
}

constexpr int FAN_THREADS = 128;
// Grid: (ceil(Nuf*Nvf / 128), n_cp); one thread per ray, lanes along a (= along u^ in the patient x-y plane).
// fan [n_cp][Nw][bh][bw] with stride fan_stride per control point.  Positions and the running sum are float64 (R1).
__global__ void __launch_bounds__(FAN_THREADS)
k_fan_depth(Params P, const CpDesc *__restrict__ desc, int n_cp, const float *__restrict__ rho, const float *__restrict__ gantry_deg,
            const float *__restrict__ zrad, const float *__restrict__ Ttab, size_t fan_stride, float *__restrict__ fan)
{
    const int cp = blockIdx.y;
    if (cp >= n_cp) return;
    const CpDesc d = desc[cp];
    if (d.a0 > d.a1) return;
    const FanBox fb = fan_box(P, d);
    const int r = blockIdx.x * FAN_THREADS + threadIdx.x;
    if (r >= fb.bw * fb.bh) return;
    const int rb = r / fb.bw, ra = r - rb * fb.bw;
    const double phi = (double)gantry_deg[cp] * 3.14159265358979323846 / 180.0;
    const double cs = cos(phi), sn = sin(phi);
    const double tu = (double)((fb.a0 + ra - P.cuf) * P.Du) / (double)P.sid, tv = (double)((fb.b0 + rb - P.cvf) * P.Dv) / (double)P.sid;
    const double dx = -sn + tu * cs, dy = cs + tu * sn, dz = tv;
    const double srcx = (double)P.isox + (double)P.sid * sn, srcy = (double)P.isoy - (double)P.sid * cs, srcz = (double)P.isoz;
    const double ds = P.ray_step;
    const int M = P.M_ray;
    // samples before the ray enters the grid's box and after it leaves contribute exact zeros: march only the samples
    // that can be inside (one sample of slack at either end: the per-sample box test decides)
    double t_in = 0.0, t_out = (double)M * ds;
    {
        const double o[3] = { (double)P.ox, (double)P.oy, (double)P.oz }, sp[3] = { (double)P.sx, (double)P.sy, (double)P.sz };
        const double s0[3] = { srcx, srcy, srcz }, dd[3] = { dx, dy, dz };
        const int N[3] = { P.nx, P.ny, P.nz };
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            if (dd[a] != 0.0) {
                const double t0 = (o[a] - 0.5 * sp[a] - s0[a]) / dd[a], t1 = (o[a] + (N[a] - 0.5) * sp[a] - s0[a]) / dd[a];
                t_in = fmax(t_in, fmin(t0, t1));
                t_out = fmin(t_out, fmax(t0, t1));
            }
        }
    }
    int m = max(0, (int)floor(t_in / ds - 0.5) - 1);
    const int m_end = min(M, (int)ceil(t_out / ds - 0.5) + 2);
    float *out = fan + (size_t)cp * fan_stride + (size_t)rb * fb.bw + ra;
    const size_t kstride = (size_t)fb.bw * fb.bh;
    const float *zc = zrad + (size_t)cp * P.Nw;
    const double inv_s[3] = { 1.0 / (double)P.sx, 1.0 / (double)P.sy, 1.0 / (double)P.sz };
    const double inv_ds = 1.0 / ds, q0 = ((double)P.sid + (double)P.wmin) * inv_ds, dq = (double)P.dw * inv_ds;   // slice k sits at q0 + k dq steps
    const float inv_dz = 1.f / P.dz;
    auto term = [&](float z) {                                  // T(z): linear between the table nodes, clamped
        const float t = z * inv_dz;
        int n0 = (int)floorf(t);
        n0 = min(max(n0, 0), P.n_z - 2);
        const float f = fminf(fmaxf(t - n0, 0.f), 1.f);
        return (1.f - f) * __ldg(Ttab + n0) + f * __ldg(Ttab + n0 + 1);
    };
    auto emit = [&](int kk, double z) {
        const float Tc = term(zc[kk]);
        out[(size_t)kk * kstride] = Tc > 0.f ? term((float)z) / Tc : 1.f;
    };
    double Z = 0.0;
    int k = 0;
    // step index m_k = min(floor(q_k), M - 1) of the next slice to emit (slices with q_k <= 0 have depth 0)
    double qk = q0;
    int mk = qk > 0.0 ? min((int)floor(qk), M - 1) : -1;
    auto next_slice = [&]() { ++k; qk = q0 + k * dq; mk = qk > 0.0 ? min((int)floor(qk), M - 1) : -1; };
    // slices in front of the first sample taken: depth 0
    while (k < P.Nw && mk < m) { emit(k, 0.0); next_slice(); }
    for (; m < m_end && k < P.Nw; ++m) {
        const double t = (m + 0.5) * ds;
        const double v = (double)density_at_f(P, rho, inv_s, srcx + t * dx, srcy + t * dy, srcz + t * dz);
        while (k < P.Nw && mk == m) { emit(k, Z + (qk - mk) * v * ds); next_slice(); }     // slices whose depth falls into this step
        Z += v * ds;
    }
    while (k < P.Nw) { emit(k, Z); next_slice(); }
}

// Multiplies vol (Phivol over S_k, forward; H_b over S_k, adjoint) by the bilinear interpolant (indices clamped to the ray
// box) of the depth factor at the voxel's sampling position (fa, fb) of Eq. 5.  Grid: (X, n_cp); a warp per (slice, row) unit.
__global__ void __launch_bounds__(256)
k_apply_fan(Params P, const CpDesc *__restrict__ desc, const SliceBox16 *__restrict__ sbox, int cp0, int n_cp, size_t fan_stride,
            const float *__restrict__ fan, float *__restrict__ vol)
{
    const int slot = blockIdx.y;
    if (slot >= n_cp) return;
    const int cp = cp0 + slot;
    const CpDesc d = desc[cp];
    if (d.a0 > d.a1) return;
    const FanBox fb = fan_box(P, d);
    const int lane = threadIdx.x & 31;
    const int warp0 = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, n_warps = (gridDim.x * blockDim.x) >> 5;
    float *vc = vol + (size_t)slot * (size_t)P.stride_cp;
    for (int q = warp0; q < P.Nw * d.pu; q += n_warps) {           // (slice, row) units of the control point's region
        const int k = q / d.pu, i = d.ri0 + (q - k * d.pu);
        const SliceBox16 S = load_box(sbox, (size_t)cp * P.Nw + k);
        if (S.u0 > S.u1 || i < S.u0 || i > S.u1) continue;
        const float mag = P.sid / (P.sid + P.wmin + k * P.dw);
        const float su = mag * P.du / P.Du, sv = mag / P.Dv;
        const float *Fk = fan + (size_t)cp * fan_stride + (size_t)k * fb.bw * fb.bh;
        const float fa = (i - P.cu) * su + P.cuf - (float)fb.a0;
        const float fla = floorf(fa);
        const float ta = fa - fla;
        const int a0 = min(max((int)fla, 0), fb.bw - 1), a1 = min(max((int)fla + 1, 0), fb.bw - 1);
        float *row = vc + ((size_t)k * d.pu + (i - d.ri0)) * d.pv - d.rj0;
        for (int j = S.v0 + lane; j <= S.v1; j += 32) {
            const float fbv = (P.v0 + j * P.dv) * sv + P.cvf - (float)fb.b0;
            const float flb = floorf(fbv);
            const float tb = fbv - flb;
            const int b0 = min(max((int)flb, 0), fb.bh - 1), b1 = min(max((int)flb + 1, 0), fb.bh - 1);
            const float f = (1.f - tb) * ((1.f - ta) * __ldg(Fk + b0 * fb.bw + a0) + ta * __ldg(Fk + b0 * fb.bw + a1)) +
                            tb * ((1.f - ta) * __ldg(Fk + b1 * fb.bw + a0) + ta * __ldg(Fk + b1 * fb.bw + a1));
            row[j] *= f;
        }
    }
}

// Expands the compact depth factors to dense [n_cp][Nw][Nvf][Nuf] maps, 0 outside the rays traced (stage tap for tests).
__global__ void k_expand_fan(Params P, const CpDesc *__restrict__ desc, int n_cp, size_t fan_stride, const float *__restrict__ fan,
                             float *__restrict__ dense)
{
    const size_t per = (size_t)P.Nw * P.Nvf * P.Nuf, n = per * n_cp;
    for (size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (size_t)gridDim.x * blockDim.x) {
        const int cp = (int)(e / per);
        const size_t r = e - (size_t)cp * per;
        const int a = (int)(r % P.Nuf), b = (int)((r / P.Nuf) % P.Nvf), k = (int)(r / ((size_t)P.Nuf * P.Nvf));
        const CpDesc &d = desc[cp];
        float v = 0.f;
        if (d.a0 <= d.a1) {
            const FanBox fb = fan_box(P, d);
            if (a >= fb.a0 && a < fb.a0 + fb.bw && b >= fb.b0 && b < fb.b0 + fb.bh)
                v = fan[(size_t)cp * fan_stride + ((size_t)k * fb.bh + (b - fb.b0)) * fb.bw + (a - fb.a0)];
        }
        dense[e] = v;
    }
}

}  // namespace pdrt
