// pdrt_plan.cuh — the planning-loop steps around the dose path, so that a whole optimisation
// iteration stays on the device: the hardware-constrained projection of PAPER.md:83-101 (Eq. 1-3, BeamValidationLayer)
// and its transposed Jacobian, the weighted-sum objective of PAPER.md:205-210 (Eq. 10; or its quadratic variant) with
// dL/dDose, jaws tracking the aperture, and the normalised-gradient step of the c5 workload.
// All of them are tiny, latency-bound kernels; every reduction has a fixed order (deterministic, no float atomics).
#pragma once
#include "pdrt_dev.cuh"

namespace pdrt {

struct PlanLimits { float leaf_w_min, leaf_F, jaw_w_min, jaw_Fx, jaw_Fy, mu_eps; };

// Eq. 1-2: centre / width of an opposing pair, minimum opening, centre clamped to the travel range, reconstruction.
__device__ __forceinline__ void validate_pair(float pa, float pb, float w_min, float F, float &qa, float &qb)
{
    float c = 0.5f * (pa + pb), w = pb - pa;
    w = fmaxf(w, w_min);
    c = fminf(fmaxf(c, -F), F);
    qa = c - 0.5f * w;
    qb = c + 0.5f * w;
}
// Transposed Jacobian of validate_pair at (pa, pb); a clamp passes the gradient where its input lies inside the closed
// interval (reading G23).
__device__ __forceinline__ void validate_pair_adjoint(float pa, float pb, float w_min, float F, float ga_hat, float gb_hat, float &ga, float &gb)
{
    const float c = 0.5f * (pa + pb), w = pb - pa;
    float gc = ga_hat + gb_hat, gw = 0.5f * (gb_hat - ga_hat);
    if (!(c >= -F && c <= F)) gc = 0.f;
    if (!(w >= w_min)) gw = 0.f;
    ga = 0.5f * gc - gw;
    gb = 0.5f * gc + gw;
}

// One thread per pair: n_pairs leaf pairs + 2 jaw pairs per control point; thread (cp, n_pairs + 2) clamps MU (Eq. 3's eps).
// ADJ = false: parameters -> projected parameters.  ADJ = true: gradients w.r.t. projected -> gradients w.r.t. raw parameters.
template <bool ADJ>
__global__ void __launch_bounds__(256)
k_validate(int n_cp, int n_pairs, PlanLimits lim, const float *__restrict__ leaves, const float *__restrict__ jaws, const float *__restrict__ mu,
           const float *__restrict__ gl_hat, const float *__restrict__ gj_hat, const float *__restrict__ gm_hat,
           float *__restrict__ out_l, float *__restrict__ out_j, float *__restrict__ out_m)
{
    const int per = n_pairs + 3;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)n_cp * per) return;
    const int cp = (int)(t / per), e = (int)(t - (long long)cp * per);
    if (e < n_pairs) {
        const size_t ia = (size_t)cp * 2 * n_pairs + e, ib = ia + n_pairs;
        if (ADJ) validate_pair_adjoint(leaves[ia], leaves[ib], lim.leaf_w_min, lim.leaf_F, gl_hat[ia], gl_hat[ib], out_l[ia], out_l[ib]);
        else validate_pair(leaves[ia], leaves[ib], lim.leaf_w_min, lim.leaf_F, out_l[ia], out_l[ib]);
    } else if (e < n_pairs + 2) {
        const int q = e - n_pairs;                       // 0: (x1, x2), 1: (y1, y2)
        const size_t ia = (size_t)cp * 4 + 2 * q, ib = ia + 1;
        const float F = q == 0 ? lim.jaw_Fx : lim.jaw_Fy;
        if (ADJ) validate_pair_adjoint(jaws[ia], jaws[ib], lim.jaw_w_min, F, gj_hat[ia], gj_hat[ib], out_j[ia], out_j[ib]);
        else validate_pair(jaws[ia], jaws[ib], lim.jaw_w_min, F, out_j[ia], out_j[ib]);
    } else {
        if (ADJ) out_m[cp] = mu[cp] >= lim.mu_eps ? gm_hat[cp] : 0.f;
        else out_m[cp] = fmaxf(mu[cp], lim.mu_eps);
    }
}

constexpr int OBJ_MAX_STRUCT = 32, OBJ_THREADS = 256;
struct ObjectiveTerms { int n; int power; float lambda[OBJ_MAX_STRUCT]; float presc[OBJ_MAX_STRUCT]; };

// L = sum_s lambda_s sum_{x in s} |D(x) - p_s|^power (power 1: Eq. 10; power 2: quadratic) and g = dL/dD in one pass
// over the dose grid.  bits[x] has bit s set when voxel x belongs to structure s.  The loss is accumulated in float64:
// per thread, then per block in a fixed order; k_objective_finish adds the block partials in block order.
__global__ void __launch_bounds__(OBJ_THREADS)
k_objective(size_t n_vox, const float *__restrict__ dose, const unsigned *__restrict__ bits, ObjectiveTerms T, float *__restrict__ g,
            double *__restrict__ partial)
{
    __shared__ double red[OBJ_THREADS / 32];
    double L = 0.0;
    for (size_t x = (size_t)blockIdx.x * OBJ_THREADS + threadIdx.x; x < n_vox; x += (size_t)gridDim.x * OBJ_THREADS) {
        unsigned m = __ldg(bits + x);
        float gx = 0.f;
        if (m) {
            const float D = __ldg(dose + x);
            while (m) {
                const int s = __ffs(m) - 1;
                m &= m - 1;
                if (s < T.n) {
                    const float dlt = D - T.presc[s];
                    if (T.power == 1) { L += (double)T.lambda[s] * fabs((double)dlt); gx += dlt > 0.f ? T.lambda[s] : (dlt < 0.f ? -T.lambda[s] : 0.f); }
                    else { L += (double)T.lambda[s] * (double)dlt * (double)dlt; gx += 2.f * T.lambda[s] * dlt; }
                }
            }
        }
        g[x] = gx;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) L += __shfl_xor_sync(0xffffffffu, L, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = L;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < OBJ_THREADS / 32; ++w) s += red[w];
        partial[blockIdx.x] = s;
    }
}
__global__ void k_objective_finish(int n_partial, const double *__restrict__ partial, double *__restrict__ loss)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        double s = 0.0;
        for (int q = 0; q < n_partial; ++q) s += partial[q];
        *loss = s;
    }
}

// Jaws tracking the aperture (BASELINE.json configs[4]; recipe of DESIGN.md §4 c5): one warp per control point.  Over the
// pairs open by more than open_gap (all pairs when none is):  x1 = min l - margin, x2 = max r + margin, y1 / y2 = the
// leaf boundaries that enclose them.
__global__ void __launch_bounds__(256)
k_track_jaws(int n_cp, int n_pairs, const float *__restrict__ leaf_bounds, const float *__restrict__ leaves, float margin, float open_gap,
             float *__restrict__ jaws)
{
    const int cp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    if (cp >= n_cp) return;
    const float *lv = leaves + (size_t)cp * 2 * n_pairs;
    bool any = false;
    for (int i = lane; i < n_pairs; i += 32) any |= (lv[n_pairs + i] - lv[i]) > open_gap;
    any = __any_sync(0xffffffffu, any);
    float x1 = INFINITY, x2 = -INFINITY;
    int first = n_pairs, last = -1;
    for (int i = lane; i < n_pairs; i += 32) {
        if (any && !((lv[n_pairs + i] - lv[i]) > open_gap)) continue;
        x1 = fminf(x1, lv[i]); x2 = fmaxf(x2, lv[n_pairs + i]);
        first = min(first, i); last = max(last, i);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        x1 = fminf(x1, __shfl_xor_sync(0xffffffffu, x1, o)); x2 = fmaxf(x2, __shfl_xor_sync(0xffffffffu, x2, o));
        first = min(first, __shfl_xor_sync(0xffffffffu, first, o)); last = max(last, __shfl_xor_sync(0xffffffffu, last, o));
    }
    if (lane == 0) {
        jaws[4 * cp] = x1 - margin; jaws[4 * cp + 1] = x2 + margin;
        jaws[4 * cp + 2] = leaf_bounds[first]; jaws[4 * cp + 3] = leaf_bounds[last + 1];
    }
}

// Normalised-gradient step (DESIGN.md §4 c5): theta <- theta - step * g / max|g| per group (all leaf edges of the arc; all
// MUs); a group whose gradient is identically zero does not move.  One block: max-reduction (exact, order-free), then the update.
constexpr int STEP_THREADS = 1024;
__global__ void __launch_bounds__(STEP_THREADS)
k_plan_step(int n_leaf, int n_cp, float step_leaf, float step_mu, const float *__restrict__ g_leaves, const float *__restrict__ g_mu,
            float *__restrict__ leaves, float *__restrict__ mu)
{
    __shared__ float red[2][STEP_THREADS / 32];
    __shared__ float mx[2];
    float ml = 0.f, mm = 0.f;
    for (int e = threadIdx.x; e < n_leaf; e += STEP_THREADS) ml = fmaxf(ml, fabsf(g_leaves[e]));
    for (int e = threadIdx.x; e < n_cp; e += STEP_THREADS) mm = fmaxf(mm, fabsf(g_mu[e]));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { ml = fmaxf(ml, __shfl_xor_sync(0xffffffffu, ml, o)); mm = fmaxf(mm, __shfl_xor_sync(0xffffffffu, mm, o)); }
    if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = ml; red[1][threadIdx.x >> 5] = mm; }
    __syncthreads();
    if (threadIdx.x < 2) {
        float m = 0.f;
        for (int w = 0; w < STEP_THREADS / 32; ++w) m = fmaxf(m, red[threadIdx.x][w]);
        mx[threadIdx.x] = m;
    }
    __syncthreads();
    ml = mx[0]; mm = mx[1];
    if (ml > 0.f) for (int e = threadIdx.x; e < n_leaf; e += STEP_THREADS) leaves[e] -= step_leaf * g_leaves[e] / ml;
    if (mm > 0.f) for (int e = threadIdx.x; e < n_cp; e += STEP_THREADS) mu[e] -= step_mu * g_mu[e] / mm;
}

}  // namespace pdrt
