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
    // exclusive scan of the per-thread sums
    __shared__ double part[DEPTH_THREADS];
    part[tid] = run;
    __syncthreads();
    if (tid == 0) {
        double s = 0.0;
        for (int q = 0; q < DEPTH_THREADS; ++q) { const double v = part[q]; part[q] = s; s += v; }
    }
    __syncthreads();
    double z = part[tid];
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

}  // namespace pdrt
