// pdrt_engine.cu — engine object and the C ABI of include/pdrt.h.  Host code only marshals arguments,
// builds the depth-indexed kernel table once (float64 -> float32) and enqueues kernels; every step of
// the dose path runs in the kernels of pdrt_{fluence,depth,conv,resample}.cuh.  No CPU fallback.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <initializer_list>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/pdrt.h"
#include "pdrt_conv.cuh"
#include "pdrt_conv_sym.cuh"
#include "pdrt_conv_fold.cuh"
#include "pdrt_depth.cuh"
#include "pdrt_dev.cuh"
#include "pdrt_fluence.cuh"
#include "pdrt_plan.cuh"
#include "pdrt_resample.cuh"

using namespace pdrt;

namespace {

std::string g_create_error;

// compiled conv variants; a requested size k runs on the smallest KT >= k with the table embedded in zeros
const int kCompiled[] = { 5, 11, 15, 21, 25, 31, 41, 51, 55, 63, 75 };     // 75: k_conv_fold only
const int kMaxKernel = 255;            // NB = 9 passes per axis of KT = 31 at most
// The single-pass convolution runs in row-symmetric form (k_conv_sym) unless PDRT_CONV_LEGACY=1 asks for the output-stationary
// kernel (k_conv), which also serves the sub-kernel passes of a split (their off-centre blocks are not symmetric by themselves).
bool conv_legacy()
{
    const char *v = std::getenv("PDRT_CONV_LEGACY");
    return v && std::atoi(v) != 0;
}
// Kernels up to `single_max` run as one pass on the smallest compiled variant; larger ones are split into NB x NB sub-kernels of
// at most 31 taps (NB odd, so that the window stays centred): fewer multiply-adds with structural zeros than one wide pass
// (halo overhead ((s + KT - 1)/s)^2 per pass instead of ((s + K - 1)/s)^2), and no limit on K from registers or shared memory.
int conv_single_max()
{
    const int widest = conv_legacy() ? 63 : 75;      // the 75-tap variant exists as k_conv_fold only
    if (const char *v = std::getenv("PDRT_CONV_SINGLE_MAX")) { const int m = std::atoi(v); if (m >= 3 && m <= widest) return m; }
    return widest;   // measured on c4: one pass (k_conv_fold) wins up to the widest compiled variant
}
// Largest compiled size for which the ADJOINT also runs in symmetric form.  The forward shares every row correlation between two output
// rows; the adjoint only where both rows r-d and r+d lie in S_k, so it gains less on supports shorter than the kernel.  With the column
// symmetry folded in as well (k_conv_fold) it wins at every single-pass size measured; the knob stays for experiments.
int conv_sym_adj_max()
{
    if (const char *v = std::getenv("PDRT_CONV_SYM_ADJ_MAX")) return std::atoi(v);
    return 75;
}
// Largest compiled size that also folds the column symmetry (k_conv_fold; units of 4 columns up to 31 taps, of 2 above).
int conv_fold_max()
{
    if (const char *v = std::getenv("PDRT_CONV_FOLD_MAX")) return std::atoi(v);
    return 75;
}
int conv_sym_fwd_min()
{
    if (const char *v = std::getenv("PDRT_CONV_SYM_FWD_MIN")) return std::atoi(v);
    return 11;
}
int compiled_size(int k)
{
    for (int kt : kCompiled)
        if (kt >= k) return kt;
    return -1;
}
// input-tile budget of one warp: the rows spanned by 32 consecutive thread-tiles of an active area `naf` tiles wide
int tile_floats_for(int kt)
{
    int best = 0;
    for (int naf = 1; naf <= NTFC_MAX; ++naf) {
        const int spans = std::min((CONV_CHUNK_TILES + naf - 1) / naf + 1, CONV_CHUNK_TILES);
        best = std::max(best, conv_pitch(kt, naf) * (spans * RS + kt - 1));
    }
    return best;
}
// blocks per control point of k_project (a block takes every X-th slice) and of k_resample_adjoint (256 beam rows per chunk)
int project_blocks(const Params &P) { return std::max(1, std::min(P.Nw, 8)); }
int resample_adj_blocks(const Params &P) { return std::max(1, std::min(48, (P.Nw * (P.Nu + RS) + RA_THREADS - 1) / RA_THREADS)); }
size_t conv_smem_bytes(int kt) { return sizeof(float) * (2 * (size_t)(kt + 1) * ((kt + 3) & ~3) + tile_floats_for(kt)); }   // row-pair kernel + ring

template <typename T> struct DevBuf {
    T *p = nullptr;
    size_t n = 0;
    cudaError_t ensure(size_t count)
    {
        if (count <= n) return cudaSuccess;
        if (p) cudaFree(p);
        p = nullptr; n = 0;
        cudaError_t e = cudaMalloc((void **)&p, count * sizeof(T));
        if (e == cudaSuccess) n = count;
        return e;
    }
    void release() { if (p) cudaFree(p); p = nullptr; n = 0; }
    size_t bytes() const { return n * sizeof(T); }
};

}  // namespace

struct pdrt_engine {
    int device = 0, sm_count = 148;
    Params P{};
    FluTables T{};
    int K = 0;
    std::vector<double> kA, ka, kB, kb;
    std::string err;
    // persistent device data
    DevBuf<float> density, wtab, pool, ttab;
    int depth_mode = PDRT_DEPTH_AXIS;
    DevBuf<float> fan;                // PDRT_DEPTH_FAN: depth factor at the ray nodes, [n_cp][Nw][bh][bw] with stride fan_stride()
    size_t fan_stride() const { return (size_t)P.Nw * P.Nuf * P.Nvf; }
    // per-call scratch (sized by control-point capacity)
    DevBuf<CpDesc> desc;
    DevBuf<SliceBox16> sbox, wbox;     // [n_cp][Nw] per-slice boxes: fluence support S_k, written part of D_b
    DevBuf<int> tile_base;
    DevBuf<WorkCounters> counters;
    DevBuf<float> phimap, phimapT, P0, T1, T2, T3, Abuf, gphimap, zrad, gT;
    DevBuf<double> rho_s, Z_s;
    DevBuf<float> bufA, bufB;         // compact beam-frame blocks: conv output (D_b / H_b) and conv input (Phivol / G_b)
    // staging for the *_host entry points
    DevBuf<float> s_dose, s_g;
    // parameters and gradients of the host calls travel packed: one pinned host block, one copy per direction and call
    // ([0]: forward call, [1]: backward call; leaves | jaws | gantry | mu, each padded to 4 floats)
    DevBuf<float> s_par[2], s_grad;
    float *h_par[2] = { nullptr, nullptr }, *h_grad = nullptr;
    size_t h_par_n[2] = { 0, 0 }, h_grad_n = 0;
    cudaEvent_t ev_par[2] = { nullptr, nullptr };     // the packed block has left the pinned host buffer
    bool par_recorded[2] = { false, false };
    // the host variants move the two volumes on copy streams of their own, so that the dose can travel to the host while the
    // next call computes and dL/dDose can travel to the device while the backward pass sets up (PCIe is full duplex)
    cudaStream_t cs_in = nullptr, cs_out = nullptr;
    cudaEvent_t ev_fwd = nullptr, ev_out = nullptr, ev_g = nullptr, ev_bwd = nullptr;
    bool out_pending = false, bwd_recorded = false;
    // S2 (and, in the backward call, the transposition of dL/dDose) do not depend on S1: they run on a side stream beside k_fluence
    // (fork after what is queued on the call's stream, join before the first kernel that needs them); not while stage timing is on
    cudaStream_t cs_side = nullptr;
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    bool side_open = false;
    DevBuf<double> obj_partial;       // block partials of the objective
    size_t scratch_cap_bytes = (size_t)48 << 30;
    int last_n_cp = 0;
    bool last_backward = false;
    cudaStream_t last_stream = nullptr;
    int conv_grid = 0;
    bool sym_fwd = false, sym_adj = false;   // which directions run k_conv_sym / k_conv_fold (single pass, from 11 taps)
    int conv_sym_per_sm[2][64] = {};
    int conv_fold_per_sm[2][80] = {};     // the same for k_conv_sym, by [adjoint][KT]
    int conv_per_sm[2][2][2][64] = {};   // resident conv blocks per SM on THIS engine's device, by [adjoint][copy width - 1][multi-pass][KT]; 0 = not queried yet
    DevBuf<float> coll;               // collimator angles [coll_n] set by pdrt_set_collimator (coll_n = 0: none)
    int coll_n = 0;
    int nzp = 0;                      // row pitch of gT: nz rounded up to 4
    int pa_warps = 0;                 // warps of k_project_adjoint that hold a shared-memory plane (0: attribute not set yet)
    // per-stage device timing of the most recent call (CUDA events on the call's stream)
    bool profiling = false;
    struct StageRec { int stage; cudaEvent_t a, b; };
    std::vector<StageRec> recs;
    std::vector<cudaEvent_t> ev_pool;
    size_t ev_used = 0;
    int launches[PDRT_N_STAGES] = {};

    size_t scratch_bytes() const
    {
        return desc.bytes() + sbox.bytes() + wbox.bytes() + tile_base.bytes() + phimap.bytes() + phimapT.bytes() + P0.bytes() + T1.bytes() + T2.bytes() +
               T3.bytes() + Abuf.bytes() + gphimap.bytes() + zrad.bytes() + gT.bytes() + rho_s.bytes() + Z_s.bytes() + bufA.bytes() + bufB.bytes();
    }
};

namespace {

int fail(pdrt_engine *e, int code, const std::string &msg)
{
    if (e) e->err = msg; else g_create_error = msg;
    return code;
}
#define CU(e, call)                                                                                  \
    do {                                                                                             \
        cudaError_t _s = (call);                                                                     \
        if (_s != cudaSuccess)                                                                       \
            return fail((e), _s == cudaErrorMemoryAllocation ? PDRT_ENOMEM : PDRT_ECUDA,             \
                        std::string(#call) + ": " + cudaGetErrorString(_s));                         \
    } while (0)

// Brackets the kernel launches of one stage with CUDA events when profiling is on; always counts launches.
struct StageTimer {
    pdrt_engine *e; cudaStream_t st; size_t rec = (size_t)-1;
    StageTimer(pdrt_engine *e_, int stage, cudaStream_t st_, int n_launches = 1) : e(e_), st(st_)
    {
        e->launches[stage] += n_launches;
        if (!e->profiling) return;
        cudaEvent_t ev[2];
        for (int q = 0; q < 2; ++q) {
            if (e->ev_used == e->ev_pool.size()) {
                cudaEvent_t n;
                if (cudaEventCreate(&n) != cudaSuccess) return;
                e->ev_pool.push_back(n);
            }
            ev[q] = e->ev_pool[e->ev_used++];
        }
        e->recs.push_back({ stage, ev[0], ev[1] });
        rec = e->recs.size() - 1;
        cudaEventRecord(ev[0], st);
    }
    ~StageTimer() { if (rec != (size_t)-1) cudaEventRecord(e->recs[rec].b, st); }
};
void reset_stage_records(pdrt_engine *e)
{
    e->recs.clear();
    e->ev_used = 0;
    for (int q = 0; q < PDRT_N_STAGES; ++q) e->launches[q] = 0;
}

// Gaussian taps (G13): g[t] ∝ exp(-(t D)^2 / 2 sigma^2), |t| <= ceil(3 sigma / D), normalised.
int gaussian_taps(double sigma, double D, std::vector<float> &g)
{
    if (!(sigma > 0.0)) { g.assign(1, 1.f); return 0; }
    const int T = (int)std::ceil(3.0 * sigma / D);
    std::vector<double> w(2 * T + 1);
    double sum = 0.0;
    for (int t = -T; t <= T; ++t) { w[t + T] = std::exp(-0.5 * (t * D / sigma) * (t * D / sigma)); sum += w[t + T]; }
    g.resize(2 * T + 1);
    for (int t = 0; t <= 2 * T; ++t) g[t] = (float)(w[t] / sum);
    return T;
}

// Pencil-kernel table (G3, G4): pixel-integrated weights of
// K(r;z) = (A e^{-a r} + B e^{-b r}) / r  by 8x8 midpoint sub-sampling, one quadrant computed and mirrored,
// embedded centred in the compiled KT x KT window.  Device layout: [n_z][KT (du)][KP (dv)], KP = KT rounded up to 4,
// i.e. exactly the shared-memory image the conv kernel wants.  The table is point-symmetric (mirrored quadrant), so the
// flipped kernel of the adjoint is the same table (R3).
// The work-item layout (chunk width, written box of D_b) follows the kernel that runs in this direction; k_fluence tabulates it per call.
void set_conv_direction(pdrt_engine *e, bool adjoint)
{
    e->P.conv_sym = (adjoint ? e->sym_adj : e->sym_fwd) ? (e->P.KT >= 15 && e->P.KT <= conv_fold_max() ? 2 : 1) : 0;   // measured: the fold pays from 15 taps
    e->P.ntfc_max = e->P.conv_sym == 2 ? fold_cols_max(e->P.KT) / 8 : e->P.conv_sym ? SYM_NTFC_MAX : NTFC_MAX;
}

int build_kernel_table(pdrt_engine *e, int k)
{
    int nb = 1, kt = compiled_size(k);
    if (k > conv_single_max()) {
        nb = 3;
        while ((k + nb - 1) / nb > 31) nb += 2;
        kt = compiled_size(((k + nb - 1) / nb) | 1);
    }
    const int T = nb * kt;                              // odd: the K x K kernel sits centred in the T x T window
    const int c = (k - 1) / 2, cT = (T - 1) / 2, nz = e->P.n_z;
    const double du = e->P.du, dv = e->P.dv;
    const int kp = (kt + 3) & ~3;
    const size_t blk = (size_t)nz * kt * kp;
    std::vector<float> tab(blk * nb * nb, 0.f);
    std::vector<double> rad((size_t)(c + 1) * (c + 1) * 64);
    for (int qj = 0; qj <= c; ++qj)
        for (int qi = 0; qi <= c; ++qi)
            for (int sj = 0; sj < 8; ++sj)
                for (int si = 0; si < 8; ++si) {
                    const double x = (qi + (si + 0.5) / 8.0 - 0.5) * du, y = (qj + (sj + 0.5) / 8.0 - 0.5) * dv;
                    rad[(((size_t)qj * (c + 1) + qi) * 8 + sj) * 8 + si] = std::sqrt(x * x + y * y);
                }
    // window position (wi along u, wj along v) -> block (wi / kt, wj / kt), image [du][dv padded to kp] of that block
    auto at = [&](int n, int wi, int wj) -> float & {
        return tab[(size_t)((wi / kt) * nb + (wj / kt)) * blk + (size_t)n * kt * kp + (size_t)(wi % kt) * kp + (wj % kt)];
    };
    for (int n = 0; n < nz; ++n) {
        const double A = e->kA[n], a = e->ka[n], B = e->kB[n], b = e->kb[n];
        for (int qj = 0; qj <= c; ++qj)
            for (int qi = 0; qi <= c; ++qi) {
                double s = 0.0;
                const double *r = &rad[((size_t)qj * (c + 1) + qi) * 64];
                for (int q = 0; q < 64; ++q) s += (A * std::exp(-a * r[q]) + B * std::exp(-b * r[q])) / r[q];
                const float w = (float)(s * du * dv / 64.0);
                at(n, cT + qi, cT + qj) = w; at(n, cT + qi, cT - qj) = w;
                at(n, cT - qi, cT + qj) = w; at(n, cT - qi, cT - qj) = w;
            }
    }
    CU(e, e->wtab.ensure(tab.size()));
    CU(e, cudaMemcpy(e->wtab.p, tab.data(), tab.size() * sizeof(float), cudaMemcpyHostToDevice));
    e->K = k;
    e->P.K = k;
    e->P.KT = kt;
    e->P.NB = nb;
    e->P.CH = c;
    e->P.tile_floats = tile_floats_for(kt);
    e->sym_fwd = nb == 1 && !conv_legacy() && kt >= conv_sym_fwd_min();
    e->sym_adj = nb == 1 && !conv_legacy() && kt >= conv_sym_fwd_min() && kt <= conv_sym_adj_max();
    set_conv_direction(e, false);
    return PDRT_OK;
}

template <int KT, bool ADJ, int CPL, bool MULTI>
int launch_conv_pass(pdrt_engine *e, int cp0, int n, const float *wtab, const float *in, float *out, const ConvPass &pass, cudaStream_t st)
{
    static_assert(KT < 64, "conv_per_sm is indexed by KT");
    int &per_sm = e->conv_per_sm[ADJ ? 1 : 0][CPL - 1][MULTI ? 1 : 0][KT];   // per engine (= per device): the opt-in attribute is a per-device setting
    const size_t smem = conv_smem_bytes(KT);
    if (per_sm == 0) {
        CU(e, cudaFuncSetAttribute(k_conv<KT, ADJ, CPL, MULTI>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int n_res = 0;
        CU(e, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n_res, k_conv<KT, ADJ, CPL, MULTI>, CONV_THREADS, smem));
        per_sm = n_res < 1 ? 1 : n_res;
    }
    e->conv_grid = e->sm_count * per_sm;              // persistent grid: a multiple of the SM count
    k_conv<KT, ADJ, CPL, MULTI><<<e->conv_grid, CONV_THREADS, smem, st>>>(e->P, e->desc.p, cp0, n, e->tile_base.p, e->zrad.p, wtab, in, out,
                                                                         e->tile_base.p + n + 1, pass);
    CU(e, cudaGetLastError());
    return PDRT_OK;
}
template <int KT, bool ADJ>
int launch_conv_fold(pdrt_engine *e, int cp0, int n, const float *in, float *out, cudaStream_t st)
{
    int &per_sm = e->conv_fold_per_sm[ADJ ? 1 : 0][KT];
    const size_t smem = fold_smem_bytes(KT);
    if (per_sm == 0) {
        CU(e, cudaFuncSetAttribute(k_conv_fold<KT, ADJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int n_res = 0;
        CU(e, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n_res, k_conv_fold<KT, ADJ>, CONV_THREADS, smem));
        per_sm = n_res < 1 ? 1 : n_res;
    }
    e->conv_grid = e->sm_count * per_sm;              // persistent grid: a multiple of the SM count
    k_conv_fold<KT, ADJ><<<e->conv_grid, CONV_THREADS, smem, st>>>(e->P, e->desc.p, cp0, n, e->tile_base.p, e->zrad.p, e->wtab.p, in, out,
                                                                   e->tile_base.p + n + 1, e->counters.p, fold_in_floats(KT), fold_out_floats(KT));
    CU(e, cudaGetLastError());
    return PDRT_OK;
}
template <int KT, bool ADJ>
int launch_conv_sym(pdrt_engine *e, int cp0, int n, const float *in, float *out, cudaStream_t st)
{
    if constexpr (KT >= 15) {
        if (e->P.conv_sym == 2) return launch_conv_fold<KT, ADJ>(e, cp0, n, in, out, st);
    }
    int &per_sm = e->conv_sym_per_sm[ADJ ? 1 : 0][KT];
    const size_t smem = sym_smem_bytes(KT);
    if (per_sm == 0) {
        CU(e, cudaFuncSetAttribute(k_conv_sym<KT, ADJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        int n_res = 0;
        CU(e, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n_res, k_conv_sym<KT, ADJ>, CONV_THREADS, smem));
        per_sm = n_res < 1 ? 1 : n_res;
    }
    e->conv_grid = e->sm_count * per_sm;              // persistent grid: a multiple of the SM count
    k_conv_sym<KT, ADJ><<<e->conv_grid, CONV_THREADS, smem, st>>>(e->P, e->desc.p, cp0, n, e->tile_base.p, e->zrad.p, e->wtab.p, in, out,
                                                                  e->tile_base.p + n + 1, e->counters.p, sym_in_floats(KT), sym_out_floats(KT));
    CU(e, cudaGetLastError());
    return PDRT_OK;
}
// All NB x NB passes of one convolution, the centre block first (it writes; the others accumulate).  Returns the launches made.
template <int KT, bool ADJ>
int launch_conv_t(pdrt_engine *e, int cp0, int n, const float *in, float *out, cudaStream_t st)
{
    if (e->P.conv_sym) return launch_conv_sym<KT, ADJ>(e, cp0, n, in, out, st);
    const int nb = e->P.NB, nbh = (nb - 1) / 2, C = (KT - 1) / 2;
    const size_t blk = (size_t)e->P.n_z * KT * ((KT + 3) & ~3);
    bool first = true;
    for (int pi = 0; pi < nb * nb; ++pi) {
        // visit order: centre block, then the rest
        const int centre = nbh * nb + nbh;
        const int q = pi == 0 ? centre : (pi <= centre ? pi - 1 : pi);
        const int bi = q / nb, bj = q % nb;
        const ConvPass pass{ (bi - nbh) * KT, (bj - nbh) * KT, first ? 1 : 0 };
        if (!first) CU(e, cudaMemsetAsync(e->tile_base.p + n + 1, 0, sizeof(int), st));      // the unit counter of the next pass
        const float *wt = e->wtab.p + (size_t)q * blk;
        int rc;
        if constexpr (KT <= 31) {                     // sub-kernels of a split have at most 31 taps
            if (nb > 1)
                rc = ((C - pass.sv) % 2 == 0) ? launch_conv_pass<KT, ADJ, 2, true>(e, cp0, n, wt, in, out, pass, st)
                                              : launch_conv_pass<KT, ADJ, 1, true>(e, cp0, n, wt, in, out, pass, st);
            else
                rc = launch_conv_pass<KT, ADJ, (C % 2 == 0) ? 2 : 1, false>(e, cp0, n, wt, in, out, pass, st);
        } else {
            if (nb > 1) return fail(e, PDRT_EINVAL, "sub-kernels of a split convolution have at most 31 taps");
            rc = launch_conv_pass<KT, ADJ, (C % 2 == 0) ? 2 : 1, false>(e, cp0, n, wt, in, out, pass, st);
        }
        if (rc) return rc;
        first = false;
    }
    return PDRT_OK;
}
template <bool ADJ> int launch_conv(pdrt_engine *e, int cp0, int n, const float *in, float *out, cudaStream_t st)
{
    switch (e->P.KT) {
    case 5: return launch_conv_t<5, ADJ>(e, cp0, n, in, out, st);
    case 11: return launch_conv_t<11, ADJ>(e, cp0, n, in, out, st);
    case 15: return launch_conv_t<15, ADJ>(e, cp0, n, in, out, st);
    case 21: return launch_conv_t<21, ADJ>(e, cp0, n, in, out, st);
    case 25: return launch_conv_t<25, ADJ>(e, cp0, n, in, out, st);
    case 31: return launch_conv_t<31, ADJ>(e, cp0, n, in, out, st);
    case 41: return launch_conv_t<41, ADJ>(e, cp0, n, in, out, st);
    case 51: return launch_conv_t<51, ADJ>(e, cp0, n, in, out, st);
    case 55: return launch_conv_t<55, ADJ>(e, cp0, n, in, out, st);
    case 63: return launch_conv_t<63, ADJ>(e, cp0, n, in, out, st);
    case 75: if (e->P.conv_sym == 2) return launch_conv_fold<75, ADJ>(e, cp0, n, in, out, st); break;
    }
    return fail(e, PDRT_EINVAL, "no compiled convolution variant for this kernel size");
}

int ensure_cp_scratch(pdrt_engine *e, int n_cp)
{
    const size_t nmap = (size_t)n_cp * e->P.Nuf * e->P.Nvf;
    CU(e, e->desc.ensure(n_cp));
    CU(e, e->sbox.ensure((size_t)n_cp * e->P.Nw)); CU(e, e->wbox.ensure((size_t)n_cp * e->P.Nw));
    CU(e, e->tile_base.ensure((size_t)n_cp + 2));     // prefix of the conv units + the unit counter of the running conv
    CU(e, e->counters.ensure(1));
    CU(e, e->phimap.ensure(nmap)); CU(e, e->phimapT.ensure(nmap)); CU(e, e->P0.ensure(nmap)); CU(e, e->T1.ensure(nmap));
    CU(e, e->T2.ensure(nmap)); CU(e, e->Abuf.ensure(nmap));
    CU(e, e->zrad.ensure((size_t)n_cp * e->P.Nw));
    CU(e, e->rho_s.ensure((size_t)n_cp * e->P.M_ray));
    CU(e, e->Z_s.ensure((size_t)n_cp * (e->P.M_ray + 1)));
    return PDRT_OK;
}
// control points per batch so that `nbuf` compact buffers stay within the scratch cap
int batch_size(const pdrt_engine *e, int n_cp, int nbuf)
{
    const size_t per_cp = (size_t)e->P.stride_cp * sizeof(float) * nbuf;
    size_t b = e->scratch_cap_bytes / per_cp;
    if (b < 1) b = 1;
    return (int)(b < (size_t)n_cp ? b : (size_t)n_cp);
}

int check_call(pdrt_engine *e, int n_cp, std::initializer_list<const void *> ptrs, bool dose_call = true)
{
    if (!e) return fail(nullptr, PDRT_EINVAL, "null engine");
    if (n_cp < 1) return fail(e, PDRT_EINVAL, "n_cp must be >= 1");
    for (const void *p : ptrs)
        if (!p) return fail(e, PDRT_EINVAL, "null pointer argument");
    CU(e, cudaSetDevice(e->device));
    if (dose_call) reset_stage_records(e);          // the planning-loop calls keep the stage records of the last dose call
    return PDRT_OK;
}

// S1 + descriptors for all control points, S2 depths
// Side stream: opened after everything queued on `st` so far, closed (joined) before the first kernel that needs its results.
int side_fork(pdrt_engine *e, cudaStream_t st)
{
    if (!e->cs_side) {
        CU(e, cudaStreamCreateWithFlags(&e->cs_side, cudaStreamNonBlocking));
        CU(e, cudaEventCreateWithFlags(&e->ev_fork, cudaEventDisableTiming));
        CU(e, cudaEventCreateWithFlags(&e->ev_join, cudaEventDisableTiming));
    }
    CU(e, cudaEventRecord(e->ev_fork, st));
    CU(e, cudaStreamWaitEvent(e->cs_side, e->ev_fork, 0));
    e->side_open = true;
    return PDRT_OK;
}
int side_join(pdrt_engine *e, cudaStream_t st)
{
    if (!e->side_open) return PDRT_OK;
    CU(e, cudaEventRecord(e->ev_join, e->cs_side));
    CU(e, cudaStreamWaitEvent(st, e->ev_join, 0));
    e->side_open = false;
    return PDRT_OK;
}

int run_setup(pdrt_engine *e, int n_cp, const float *leaves, const float *jaws, const float *gantry, const float *mu,
              bool need_depth, cudaStream_t st, bool defer_join = false)
{
    int rc = ensure_cp_scratch(e, n_cp);
    if (rc) return rc;
    if (e->coll_n != 0 && e->coll_n != n_cp) return fail(e, PDRT_EINVAL, "collimator angles were set for a different number of control points");
    const bool fan = e->depth_mode == PDRT_DEPTH_FAN;
    const bool beside = need_depth && !fan && !e->profiling;       // k_depth beside k_fluence (the fan marcher needs both their results)
    if (beside) {
        if ((rc = side_fork(e, st))) return rc;
        ++e->launches[PDRT_STAGE_DEPTH];
        k_depth<<<n_cp, DEPTH_THREADS, 0, e->cs_side>>>(e->P, n_cp, e->density.p, gantry, e->rho_s.p, e->Z_s.p, e->zrad.p);
        CU(e, cudaGetLastError());
    }
    {
        StageTimer t(e, PDRT_STAGE_FLUENCE, st);
        k_fluence<<<n_cp, FLU_THREADS, 0, st>>>(e->P, e->T, n_cp, leaves, jaws, gantry, e->coll_n ? e->coll.p : nullptr, mu, e->desc.p, e->sbox.p, e->wbox.p,
                                               e->P0.p, e->T1.p, e->T2.p, e->Abuf.p, e->phimap.p, e->phimapT.p);
    }
    CU(e, cudaGetLastError());
    if (need_depth && !beside) {
        if (fan) CU(e, e->fan.ensure((size_t)n_cp * e->fan_stride()));
        StageTimer t(e, PDRT_STAGE_DEPTH, st, fan ? 2 : 1);
        k_depth<<<n_cp, DEPTH_THREADS, 0, st>>>(e->P, n_cp, e->density.p, gantry, e->rho_s.p, e->Z_s.p, e->zrad.p);
        if (fan)
            k_fan_depth<<<dim3((e->P.Nuf * e->P.Nvf + FAN_THREADS - 1) / FAN_THREADS, n_cp), FAN_THREADS, 0, st>>>(
                e->P, e->desc.p, n_cp, e->density.p, gantry, e->zrad.p, e->ttab.p, e->fan_stride(), e->fan.p);
    }
    CU(e, cudaGetLastError());
    if (!defer_join && (rc = side_join(e, st))) return rc;
    return PDRT_OK;
}

int forward_impl(pdrt_engine *e, int n_cp, const float *leaves, const float *jaws, const float *gantry, const float *mu,
                 float *dose, cudaStream_t st)
{
    set_conv_direction(e, false);
    int rc = run_setup(e, n_cp, leaves, jaws, gantry, mu, true, st);
    if (rc) return rc;
    const int nb = batch_size(e, n_cp, 2);
    CU(e, e->bufA.ensure((size_t)nb * e->P.stride_cp));
    CU(e, e->bufB.ensure((size_t)nb * e->P.stride_cp));
    const dim3 gg((e->P.nx + GD_PX - 1) / GD_PX, (e->P.ny + GD_PY - 1) / GD_PY, 1);
    // the resampler writes only the z-range that the control points reach; the rest of the grid is zero
    CU(e, cudaMemsetAsync(dose, 0, sizeof(float) * (size_t)e->P.nx * e->P.ny * e->P.nz, st));
    for (int cp0 = 0; cp0 < n_cp; cp0 += nb) {
        const int n = std::min(nb, n_cp - cp0);
        {
            StageTimer t(e, PDRT_STAGE_SCAN, st);
            k_scan_items<<<1, 256, 0, st>>>(e->desc.p, cp0, n, 0, e->P.Nuf, e->P.Nvf, e->tile_base.p, e->counters.p);
        }
        CU(e, cudaGetLastError());
        {
            StageTimer t(e, PDRT_STAGE_PROJECT, st);
            k_project<<<dim3(project_blocks(e->P), n), PROJECT_THREADS, 0, st>>>(e->P, e->desc.p, e->sbox.p, cp0, n, e->phimapT.p, e->bufB.p);
            if (e->depth_mode == PDRT_DEPTH_FAN)
                k_apply_fan<<<dim3(32, n), 256, 0, st>>>(e->P, e->desc.p, e->sbox.p, cp0, n, e->fan_stride(), e->fan.p, e->bufB.p);
        }
        CU(e, cudaGetLastError());
        {
            StageTimer t(e, PDRT_STAGE_CONV, st, e->P.NB * e->P.NB);
            rc = launch_conv<false>(e, cp0, n, e->bufB.p, e->bufA.p, st);
        }
        if (rc) return rc;
        {
            StageTimer t(e, PDRT_STAGE_GATHER, st);
            k_gather_dose<<<gg, GD_THREADS, 0, st>>>(e->P, e->desc.p, e->wbox.p, cp0, n, e->bufA.p, dose, cp0 > 0);
        }
        CU(e, cudaGetLastError());
    }
    e->last_n_cp = n_cp; e->last_backward = false; e->last_stream = st;
    return PDRT_OK;
}

// S7-S9 for all control points: leaves dL/dPhimap (per control point, inside its support bbox) in e->gphimap
int backward_to_fluence(pdrt_engine *e, int n_cp, const float *leaves, const float *jaws, const float *gantry,
                        const float *mu, const float *gdose, cudaStream_t st, cudaEvent_t gdose_ready = nullptr)
{
    set_conv_direction(e, true);
    int rc = run_setup(e, n_cp, leaves, jaws, gantry, mu, true, st, true);
    if (rc) return rc;
    // S1 / S2 above do not read dL/dDose; its transposition runs on the side stream too when one is open
    cudaStream_t ts = e->side_open ? e->cs_side : st;
    if (gdose_ready) CU(e, cudaStreamWaitEvent(ts, gdose_ready, 0));
    const size_t nmap = (size_t)n_cp * e->P.Nuf * e->P.Nvf;
    CU(e, e->gphimap.ensure(nmap));
    CU(e, e->T3.ensure(nmap));
    const size_t nxy = (size_t)e->P.nx * e->P.ny;
    CU(e, e->gT.ensure(nxy * e->nzp));
    {   // S7 prologue: dL/dDose with z fastest, so that the resampling adjoint streams along v
        StageTimer t(e, PDRT_STAGE_TRANSPOSE, st);
        k_transpose_g<<<dim3((unsigned)((nxy + 31) / 32), (e->nzp + 31) / 32), 256, 0, ts>>>((int)nxy, e->P.nz, e->nzp, gdose, e->gT.p);
    }
    CU(e, cudaGetLastError());
    if ((rc = side_join(e, st))) return rc;
    if (e->pa_warps == 0) {   // planes of k_project_adjoint: as many of its 8 warps as fit into shared memory (opt-in above 48 KB, per device)
        const size_t per_warp = sizeof(float) * 32 * (size_t)e->P.Nuf;
        const int fit = (int)std::min<size_t>(PA_WARPS, (size_t)(200 << 10) / per_warp);
        if (fit < 1) return fail(e, PDRT_EINVAL, "fluence map too wide for the projection adjoint (flu_nu > 1600)");
        CU(e, cudaFuncSetAttribute(k_project_adjoint, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(per_warp * fit)));
        e->pa_warps = fit;
    }
    CU(e, cudaGetLastError());
    const int nb = batch_size(e, n_cp, 2);
    CU(e, e->bufA.ensure((size_t)nb * e->P.stride_cp));
    CU(e, e->bufB.ensure((size_t)nb * e->P.stride_cp));
    for (int cp0 = 0; cp0 < n_cp; cp0 += nb) {
        const int n = std::min(nb, n_cp - cp0);
        {
            StageTimer t(e, PDRT_STAGE_SCAN, st);
            k_scan_items<<<1, 256, 0, st>>>(e->desc.p, cp0, n, 1, e->P.Nuf, e->P.Nvf, e->tile_base.p, e->counters.p);
        }
        CU(e, cudaGetLastError());
        {
            StageTimer t(e, PDRT_STAGE_RESAMPLE_ADJ, st);
            k_resample_adjoint<<<dim3(resample_adj_blocks(e->P), n), RA_THREADS, 0, st>>>(e->P, e->desc.p, e->sbox.p, cp0, n, e->P.CH, e->nzp,
                                                                                          e->gT.p, e->bufB.p);
        }
        CU(e, cudaGetLastError());
        {
            StageTimer t(e, PDRT_STAGE_CONV_ADJ, st, e->P.NB * e->P.NB);
            rc = launch_conv<true>(e, cp0, n, e->bufB.p, e->bufA.p, st);
        }
        if (rc) return rc;
        {
            StageTimer t(e, PDRT_STAGE_PROJECT_ADJ, st);
            if (e->depth_mode == PDRT_DEPTH_FAN)      // the factor is a fixed diagonal weighting: the transpose applies it to H_b
                k_apply_fan<<<dim3(32, n), 256, 0, st>>>(e->P, e->desc.p, e->sbox.p, cp0, n, e->fan_stride(), e->fan.p, e->bufA.p);
            k_project_adjoint<<<dim3(PA_CLUSTER * ((e->P.Nvf + 31) / 32), n), PA_THREADS, sizeof(float) * 32 * (size_t)e->P.Nuf * e->pa_warps, st>>>(
                e->P, e->desc.p, e->sbox.p, cp0, n, e->pa_warps, e->bufA.p, e->gphimap.p);
        }
        CU(e, cudaGetLastError());
    }
    return PDRT_OK;
}

int backward_impl(pdrt_engine *e, int n_cp, const float *leaves, const float *jaws, const float *gantry, const float *mu,
                  const float *gdose, float *d_leaves, float *d_jaws, float *d_mu, cudaStream_t st, cudaEvent_t gdose_ready = nullptr)
{
    int rc = backward_to_fluence(e, n_cp, leaves, jaws, gantry, mu, gdose, st, gdose_ready);
    if (rc) return rc;
    {
        StageTimer t(e, PDRT_STAGE_FLUENCE_ADJ, st);
        k_fluence_adjoint<<<n_cp, FLU_THREADS, 0, st>>>(e->P, e->T, n_cp, leaves, jaws, e->desc.p, e->phimap.p, e->Abuf.p,
                                                       e->gphimap.p, e->T1.p, e->T2.p, e->T3.p, d_leaves, d_jaws, d_mu);
    }
    CU(e, cudaGetLastError());
    e->last_n_cp = n_cp; e->last_backward = true; e->last_stream = st;
    return PDRT_OK;
}

}  // namespace

extern "C" {

const char *pdrt_last_error(const pdrt_engine *engine) { return engine ? engine->err.c_str() : g_create_error.c_str(); }

int pdrt_create(const pdrt_grid *grid, const float *density, const pdrt_beam_model *m, pdrt_engine **out)
{
    if (!grid || !density || !m || !out) return fail(nullptr, PDRT_EINVAL, "null argument");
    *out = nullptr;
    if (grid->nx < 1 || grid->ny < 1 || grid->nz < 1 || !(grid->sx > 0) || !(grid->sy > 0) || !(grid->sz > 0))
        return fail(nullptr, PDRT_EINVAL, "grid sizes and spacings must be positive");
    if ((long long)grid->nx * grid->ny * grid->nz > (1ll << 31) - 1) return fail(nullptr, PDRT_EINVAL, "grid too large");
    if (grid->nx > 16384 || grid->ny > 16384 || grid->nz > 16384 || m->beam_nu > 16384 || m->beam_nw > 16384)
        return fail(nullptr, PDRT_EINVAL, "grid dimensions above 16384 are not supported");
    if (!(m->sid_mm > 0)) return fail(nullptr, PDRT_EINVAL, "sid_mm must be positive");
    if (m->n_pairs < 1 || !m->leaf_bounds_mm) return fail(nullptr, PDRT_EINVAL, "n_pairs >= 1 and leaf_bounds_mm required");
    for (int i = 0; i < m->n_pairs; ++i)
        if (!(m->leaf_bounds_mm[i] < m->leaf_bounds_mm[i + 1])) return fail(nullptr, PDRT_EINVAL, "leaf_bounds_mm must be strictly ascending");
    if (m->flu_nu < 1 || m->flu_nv < 1 || !(m->flu_du > 0) || !(m->flu_dv > 0)) return fail(nullptr, PDRT_EINVAL, "bad fluence map geometry");
    if (!(m->tau >= 0.f && m->tau <= 1.f)) return fail(nullptr, PDRT_EINVAL, "tau must lie in [0,1]");
    if (!(m->fwhm_mlc_mm >= 0) || !(m->fwhm_jaw_mm >= 0)) return fail(nullptr, PDRT_EINVAL, "penumbra FWHM must be >= 0");
    if (m->n_hs < 0 || m->n_hs > MAX_HS || (m->n_hs > 0 && (!m->hs_amp || !m->hs_sigma_mm)))
        return fail(nullptr, PDRT_EINVAL, "n_hs must lie in 0..4 with both tables given");
    if (m->n_oar < 0 || (m->n_oar > 0 && (!m->oar || !(m->oar_dr_mm > 0)))) return fail(nullptr, PDRT_EINVAL, "bad off-axis table");
    if (m->n_z < 2 || !(m->dz_mm > 0) || !m->kA || !m->ka || !m->kB || !m->kb) return fail(nullptr, PDRT_EINVAL, "kernel tables need n_z >= 2 and dz_mm > 0");
    for (int n = 0; n < m->n_z; ++n)
        if (!std::isfinite(m->kA[n]) || !std::isfinite(m->ka[n]) || !std::isfinite(m->kB[n]) || !std::isfinite(m->kb[n]))
            return fail(nullptr, PDRT_EINVAL, "non-finite kernel table entry");
    if (m->kernel_size < 3 || m->kernel_size > kMaxKernel || m->kernel_size % 2 == 0) return fail(nullptr, PDRT_EINVAL, "kernel_size must be odd, 3..255");
    if (m->beam_nu < 0 || (m->beam_nu > 0 && (m->beam_nw < 1 || !(m->beam_du > 0) || !(m->beam_dw > 0))))
        return fail(nullptr, PDRT_EINVAL, "bad beam grid");
    if (!(m->ray_step_mm >= 0)) return fail(nullptr, PDRT_EINVAL, "ray_step_mm must be >= 0");

    pdrt_engine *e = new (std::nothrow) pdrt_engine();
    if (!e) return fail(nullptr, PDRT_ENOMEM, "out of host memory");
    auto bail = [&](int code) { g_create_error = e->err; pdrt_destroy(e); return code; };
    cudaError_t s = cudaGetDevice(&e->device);
    if (s != cudaSuccess) { fail(e, PDRT_ECUDA, std::string("no CUDA device: ") + cudaGetErrorString(s)); return bail(PDRT_ECUDA); }
    cudaDeviceProp prop;
    s = cudaGetDeviceProperties(&prop, e->device);
    if (s != cudaSuccess) { fail(e, PDRT_ECUDA, std::string("cudaGetDeviceProperties: ") + cudaGetErrorString(s)); return bail(PDRT_ECUDA); }
    e->sm_count = prop.multiProcessorCount;
    if (const char *cap = std::getenv("PDRT_SCRATCH_GB")) {
        const double gb = std::atof(cap);
        if (gb > 0) e->scratch_cap_bytes = (size_t)(gb * (double)(1ull << 30));
    }
    {   // leave headroom on smaller devices
        size_t free_b = 0, total_b = 0;
        if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess && e->scratch_cap_bytes > free_b / 2) e->scratch_cap_bytes = free_b / 2;
    }

    Params &P = e->P;
    P.nx = grid->nx; P.ny = grid->ny; P.nz = grid->nz;
    P.sx = grid->sx; P.sy = grid->sy; P.sz = grid->sz;
    P.ox = grid->ox; P.oy = grid->oy; P.oz = grid->oz;
    P.isox = grid->iso[0]; P.isoy = grid->iso[1]; P.isoz = grid->iso[2];
    if (m->beam_nu > 0) { P.Nu = m->beam_nu; P.Nw = m->beam_nw; P.du = m->beam_du; P.dw = m->beam_dw; P.wmin = m->beam_wmin; }
    else { P.Nu = grid->nx; P.Nw = grid->ny; P.du = P.dw = grid->sx; P.wmin = -0.5f * (P.Nw - 1) * P.dw; }
    P.Nv = grid->nz; P.dv = grid->sz;
    e->nzp = (grid->nz + 3) & ~3;
    P.cu = 0.5f * (P.Nu - 1); P.v0 = grid->oz - grid->iso[2];
    P.Nuf = m->flu_nu; P.Nvf = m->flu_nv; P.Du = m->flu_du; P.Dv = m->flu_dv;
    P.cuf = 0.5f * (P.Nuf - 1); P.cvf = 0.5f * (P.Nvf - 1);
    P.sid = m->sid_mm; P.tau = m->tau; P.cal = m->cal; P.Np = m->n_pairs;
    P.n_z = m->n_z; P.dz = m->dz_mm;
    if (!(P.sid + P.wmin > 0)) { fail(e, PDRT_EINVAL, "beam grid must lie in front of the source (sid + beam_wmin > 0)"); return bail(PDRT_EINVAL); }
    P.ray_step = m->ray_step_mm > 0 ? (double)m->ray_step_mm : 0.5 * (double)std::fmin(grid->sx, std::fmin(grid->sy, grid->sz));
    const double dmax = (double)P.sid + (double)P.wmin + (P.Nw - 1) * (double)P.dw;
    P.M_ray = (int)std::floor(dmax / P.ray_step) + 2;
    P.stride_cp = (long long)(P.Nu + 4) * P.Nw * ((P.Nv + 7) / 8 * 8 + 16);   // bound of pu * Nw * pv, multiple of 8
    e->kA.assign(m->kA, m->kA + m->n_z); e->ka.assign(m->ka, m->ka + m->n_z);
    e->kB.assign(m->kB, m->kB + m->n_z); e->kb.assign(m->kb, m->kb + m->n_z);

    // fluence tables: one float pool on the device
    std::vector<float> pool;
    auto push = [&](const float *src, size_t n) { size_t off = pool.size(); pool.insert(pool.end(), src, src + n); while (pool.size() % 4) pool.push_back(0.f); return off; };
    const size_t o_lb = push(m->leaf_bounds_mm, m->n_pairs + 1);
    const float one = 1.f;
    const size_t o_oar = m->n_oar > 0 ? push(m->oar, m->n_oar) : push(&one, 1);
    std::vector<float> gu, gv, hgu[MAX_HS], hgv[MAX_HS];
    FluTables &T = e->T;
    T.Tu = gaussian_taps(m->fwhm_mlc_mm / 2.354820045, m->flu_du, gu);
    T.Tv = gaussian_taps(m->fwhm_jaw_mm / 2.354820045, m->flu_dv, gv);
    int tu_max = T.Tu, tv_max = T.Tv;
    size_t o_hgu[MAX_HS] = {}, o_hgv[MAX_HS] = {};
    T.n_hs = m->n_hs;
    for (int q = 0; q < m->n_hs; ++q) {
        T.hs_amp[q] = m->hs_amp[q];
        T.hs_Tu[q] = gaussian_taps(m->hs_sigma_mm[q], m->flu_du, hgu[q]);
        T.hs_Tv[q] = gaussian_taps(m->hs_sigma_mm[q], m->flu_dv, hgv[q]);
        tu_max = std::max(tu_max, T.hs_Tu[q]); tv_max = std::max(tv_max, T.hs_Tv[q]);
    }
    if (tu_max > MAX_TAPS || tv_max > MAX_TAPS) { fail(e, PDRT_EINVAL, "Gaussian wider than 64 pixels"); return bail(PDRT_EINVAL); }
    const size_t o_gu = push(gu.data(), gu.size()), o_gv = push(gv.data(), gv.size());
    for (int q = 0; q < m->n_hs; ++q) { o_hgu[q] = push(hgu[q].data(), hgu[q].size()); o_hgv[q] = push(hgv[q].data(), hgv[q].size()); }
    P.Tu_max = tu_max; P.Tv_max = tv_max;

    auto cuda_bail = [&](cudaError_t st, const char *what) {
        fail(e, st == cudaErrorMemoryAllocation ? PDRT_ENOMEM : PDRT_ECUDA, std::string(what) + ": " + cudaGetErrorString(st));
        return bail(st == cudaErrorMemoryAllocation ? PDRT_ENOMEM : PDRT_ECUDA);
    };
    if ((s = e->pool.ensure(pool.size())) != cudaSuccess) return cuda_bail(s, "cudaMalloc(tables)");
    if ((s = cudaMemcpy(e->pool.p, pool.data(), pool.size() * sizeof(float), cudaMemcpyHostToDevice)) != cudaSuccess) return cuda_bail(s, "cudaMemcpy(tables)");
    T.leaf_bounds = e->pool.p + o_lb; T.oar = e->pool.p + o_oar; T.n_oar = m->n_oar; T.oar_dr = m->n_oar > 0 ? m->oar_dr_mm : 1.f;
    T.gu = e->pool.p + o_gu; T.gv = e->pool.p + o_gv;
    for (int q = 0; q < m->n_hs; ++q) { T.hs_gu[q] = e->pool.p + o_hgu[q]; T.hs_gv[q] = e->pool.p + o_hgv[q]; }

    const size_t nvox = (size_t)P.nx * P.ny * P.nz;
    if ((s = e->density.ensure(nvox)) != cudaSuccess) return cuda_bail(s, "cudaMalloc(density)");
    if ((s = cudaMemcpy(e->density.p, density, nvox * sizeof(float), cudaMemcpyDefault)) != cudaSuccess) return cuda_bail(s, "cudaMemcpy(density)");
    {   // broad-beam depth term T(z) = 2 pi (A/a + B/b) at the table nodes (PDRT_DEPTH_FAN)
        std::vector<float> tt(m->n_z);
        for (int n = 0; n < m->n_z; ++n)
            tt[n] = (float)(2.0 * 3.14159265358979323846 * ((double)m->kA[n] / (double)m->ka[n] + (double)m->kB[n] / (double)m->kb[n]));
        if ((s = e->ttab.ensure(tt.size())) != cudaSuccess) return cuda_bail(s, "cudaMalloc(depth term)");
        if ((s = cudaMemcpy(e->ttab.p, tt.data(), tt.size() * sizeof(float), cudaMemcpyHostToDevice)) != cudaSuccess) return cuda_bail(s, "cudaMemcpy(depth term)");
    }
    if (m->depth_mode != PDRT_DEPTH_AXIS && m->depth_mode != PDRT_DEPTH_FAN) { fail(e, PDRT_EINVAL, "unknown depth_mode"); return bail(PDRT_EINVAL); }
    e->depth_mode = m->depth_mode;
    int rc = build_kernel_table(e, m->kernel_size);
    if (rc) return bail(rc);
    *out = e;
    return PDRT_OK;
}

void pdrt_destroy(pdrt_engine *e)
{
    if (!e) return;
    cudaSetDevice(e->device);
    cudaDeviceSynchronize();
    e->density.release(); e->wtab.release(); e->pool.release(); e->desc.release(); e->tile_base.release();
    e->ttab.release(); e->fan.release(); e->coll.release();
    e->sbox.release(); e->wbox.release();
    e->counters.release(); e->phimap.release(); e->P0.release(); e->T1.release(); e->T2.release(); e->T3.release();
    e->Abuf.release(); e->gphimap.release(); e->zrad.release(); e->rho_s.release(); e->Z_s.release();
    e->bufA.release(); e->bufB.release(); e->phimapT.release(); e->gT.release();
    e->s_dose.release(); e->s_g.release(); e->s_grad.release();
    for (int q = 0; q < 2; ++q) { e->s_par[q].release(); if (e->h_par[q]) cudaFreeHost(e->h_par[q]); if (e->ev_par[q]) cudaEventDestroy(e->ev_par[q]); }
    if (e->h_grad) cudaFreeHost(e->h_grad);
    if (e->cs_side) cudaStreamDestroy(e->cs_side);
    for (cudaEvent_t ev : { e->ev_fork, e->ev_join }) if (ev) cudaEventDestroy(ev);
    if (e->cs_in) cudaStreamDestroy(e->cs_in);
    if (e->cs_out) cudaStreamDestroy(e->cs_out);
    for (cudaEvent_t ev : { e->ev_fwd, e->ev_out, e->ev_g, e->ev_bwd }) if (ev) cudaEventDestroy(ev);
    e->obj_partial.release();
    for (cudaEvent_t ev : e->ev_pool) cudaEventDestroy(ev);
    delete e;
}

int pdrt_set_kernel_size(pdrt_engine *e, int32_t k)
{
    if (!e) return fail(nullptr, PDRT_EINVAL, "null engine");
    if (k < 3 || k > kMaxKernel || k % 2 == 0) return fail(e, PDRT_EINVAL, "kernel_size must be odd, 3..255");
    CU(e, cudaSetDevice(e->device));
    CU(e, cudaDeviceSynchronize());
    return build_kernel_table(e, k);
}

int pdrt_set_depth_mode(pdrt_engine *e, int32_t mode)
{
    if (!e) return fail(nullptr, PDRT_EINVAL, "null engine");
    if (mode != PDRT_DEPTH_AXIS && mode != PDRT_DEPTH_FAN) return fail(e, PDRT_EINVAL, "unknown depth_mode");
    e->depth_mode = mode;
    return PDRT_OK;
}

int pdrt_set_collimator(pdrt_engine *e, int32_t n_cp, const float *coll_deg, void *stream)
{
    if (!e) return fail(nullptr, PDRT_EINVAL, "null engine");
    if (n_cp < 0 || (n_cp > 0 && !coll_deg)) return fail(e, PDRT_EINVAL, "n_cp >= 0 and a pointer when n_cp > 0");
    CU(e, cudaSetDevice(e->device));
    if (n_cp > 0) {
        CU(e, e->coll.ensure(n_cp));
        CU(e, cudaMemcpyAsync(e->coll.p, coll_deg, sizeof(float) * n_cp, cudaMemcpyDefault, (cudaStream_t)stream));
    }
    e->coll_n = n_cp;
    return PDRT_OK;
}

int pdrt_get_info(const pdrt_engine *e, pdrt_info *info)
{
    if (!e || !info) return PDRT_EINVAL;
    const Params &P = e->P;
    info->nx = P.nx; info->ny = P.ny; info->nz = P.nz;
    info->beam_nu = P.Nu; info->beam_nv = P.Nv; info->beam_nw = P.Nw;
    info->beam_du = P.du; info->beam_dv = P.dv; info->beam_dw = P.dw; info->beam_wmin = P.wmin;
    info->flu_nu = P.Nuf; info->flu_nv = P.Nvf; info->n_pairs = P.Np;
    info->kernel_size = P.K; info->kernel_size_compiled = P.KT; info->kernel_passes = P.NB * P.NB;
    info->ray_step_mm = (float)P.ray_step; info->ray_samples = P.M_ray;
    info->sm_count = e->sm_count;
    info->scratch_bytes = e->scratch_bytes();
    return PDRT_OK;
}

int pdrt_get_work(pdrt_engine *e, pdrt_work *w)
{
    if (!e || !w) return fail(e, PDRT_EINVAL, "null argument");
    if (e->last_n_cp < 1 || !e->counters.p) return fail(e, PDRT_EINVAL, "no dose call has run on this engine yet");
    CU(e, cudaSetDevice(e->device));
    CU(e, cudaStreamSynchronize(e->last_stream));
    WorkCounters wc;
    CU(e, cudaMemcpy(&wc, e->counters.p, sizeof(wc), cudaMemcpyDeviceToHost));
    w->n_cp = e->last_n_cp;
    w->conv_items = wc.items; w->support_voxels = wc.support_vox; w->footprint_voxels = wc.footprint_vox;
    w->region_voxels = wc.region_vox; w->conv_macs = e->last_backward ? wc.macs_adj : wc.macs_fwd;
    w->kernel_size = e->P.K; w->kernel_size_compiled = e->P.KT;
    w->fan_rays = e->depth_mode == PDRT_DEPTH_FAN ? wc.fan_rays : 0;
    w->ray_samples = e->P.M_ray;
    w->conv_symmetric = (e->last_backward ? e->sym_adj : e->sym_fwd) ? (e->P.KT >= 15 && e->P.KT <= conv_fold_max() ? 2 : 1) : 0;
    return PDRT_OK;
}

int pdrt_set_profiling(pdrt_engine *e, int32_t enable)
{
    if (!e) return fail(nullptr, PDRT_EINVAL, "null engine");
    e->profiling = enable != 0;
    return PDRT_OK;
}

int pdrt_get_stage_ms(pdrt_engine *e, float *ms, int32_t *launches)
{
    if (!e || !ms || !launches) return fail(e, PDRT_EINVAL, "null argument");
    CU(e, cudaSetDevice(e->device));
    CU(e, cudaStreamSynchronize(e->last_stream));
    for (int q = 0; q < PDRT_N_STAGES; ++q) { ms[q] = 0.f; launches[q] = e->launches[q]; }
    for (const pdrt_engine::StageRec &r : e->recs) {
        float t = 0.f;
        CU(e, cudaEventElapsedTime(&t, r.a, r.b));
        ms[r.stage] += t;
    }
    return PDRT_OK;
}

int pdrt_dose(pdrt_engine *e, int32_t n_cp, const float *leaves, const float *jaws, const float *gantry, const float *mu,
              float *dose, void *stream)
{
    int rc = check_call(e, n_cp, { leaves, jaws, gantry, mu, dose });
    if (rc) return rc;
    return forward_impl(e, n_cp, leaves, jaws, gantry, mu, dose, (cudaStream_t)stream);
}

int pdrt_dose_backward(pdrt_engine *e, int32_t n_cp, const float *leaves, const float *jaws, const float *gantry,
                       const float *mu, const float *gdose, float *d_leaves, float *d_jaws, float *d_mu, void *stream)
{
    int rc = check_call(e, n_cp, { leaves, jaws, gantry, mu, gdose, d_leaves, d_jaws, d_mu });
    if (rc) return rc;
    return backward_impl(e, n_cp, leaves, jaws, gantry, mu, gdose, d_leaves, d_jaws, d_mu, (cudaStream_t)stream);
}

// Offsets [floats] of the packed parameter / gradient blocks: leaves | jaws | gantry (parameters only) | mu, each padded to 4 floats.
struct PackOff { size_t leaves, jaws, gantry, mu, total; };
static PackOff pack_offsets(const pdrt_engine *e, int n_cp, bool with_gantry)
{
    auto pad4 = [](size_t n) { return (n + 3) & ~(size_t)3; };
    PackOff o;
    o.leaves = 0;
    o.jaws = pad4((size_t)n_cp * 2 * e->P.Np);
    o.gantry = o.jaws + pad4((size_t)n_cp * 4);
    o.mu = with_gantry ? o.gantry + pad4(n_cp) : o.gantry;
    o.total = o.mu + pad4(n_cp);
    return o;
}
static int ensure_pinned(pdrt_engine *e, float **p, size_t *have, size_t want)
{
    if (want <= *have) return PDRT_OK;
    if (*p) cudaFreeHost(*p);
    *p = nullptr; *have = 0;
    CU(e, cudaHostAlloc((void **)p, want * sizeof(float), cudaHostAllocDefault));
    *have = want;
    return PDRT_OK;
}
// Packs the four host arrays into the pinned block `which` and sends it with ONE copy on `cs`; the device pointers come back in `dev`.
static int stage_params_in(pdrt_engine *e, int which, int n_cp, const float *leaves, const float *jaws, const float *gantry,
                           const float *mu, cudaStream_t cs, const float *(&dev)[4])
{
    const PackOff o = pack_offsets(e, n_cp, true);
    int rc = ensure_pinned(e, &e->h_par[which], &e->h_par_n[which], o.total);
    if (rc) return rc;
    CU(e, e->s_par[which].ensure(o.total));
    if (!e->ev_par[which]) CU(e, cudaEventCreateWithFlags(&e->ev_par[which], cudaEventDisableTiming));
    if (e->par_recorded[which]) CU(e, cudaEventSynchronize(e->ev_par[which]));       // the previous call's copy has read the pinned block
    float *h = e->h_par[which];
    std::memcpy(h + o.leaves, leaves, sizeof(float) * n_cp * 2 * e->P.Np);
    std::memcpy(h + o.jaws, jaws, sizeof(float) * n_cp * 4);
    std::memcpy(h + o.gantry, gantry, sizeof(float) * n_cp);
    std::memcpy(h + o.mu, mu, sizeof(float) * n_cp);
    CU(e, cudaMemcpyAsync(e->s_par[which].p, h, o.total * sizeof(float), cudaMemcpyHostToDevice, cs));
    CU(e, cudaEventRecord(e->ev_par[which], cs));
    e->par_recorded[which] = true;
    const float *d = e->s_par[which].p;
    dev[0] = d + o.leaves; dev[1] = d + o.jaws; dev[2] = d + o.gantry; dev[3] = d + o.mu;
    return PDRT_OK;
}

static int host_streams(pdrt_engine *e)
{
    if (e->cs_in) return PDRT_OK;
    CU(e, cudaStreamCreateWithFlags(&e->cs_in, cudaStreamNonBlocking));
    CU(e, cudaStreamCreateWithFlags(&e->cs_out, cudaStreamNonBlocking));
    for (cudaEvent_t *ev : { &e->ev_fwd, &e->ev_out, &e->ev_g, &e->ev_bwd }) CU(e, cudaEventCreateWithFlags(ev, cudaEventDisableTiming));
    return PDRT_OK;
}

int pdrt_dose_host_async(pdrt_engine *e, int32_t n_cp, const float *leaves, const float *jaws, const float *gantry,
                         const float *mu, float *dose, void *stream)
{
    int rc = check_call(e, n_cp, { leaves, jaws, gantry, mu, dose });
    if (rc) return rc;
    if ((rc = host_streams(e))) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nvox = (size_t)e->P.nx * e->P.ny * e->P.nz;
    const float *par[4];
    if ((rc = stage_params_in(e, 0, n_cp, leaves, jaws, gantry, mu, st, par))) return rc;
    CU(e, e->s_dose.ensure(nvox));
    if (e->out_pending) CU(e, cudaStreamWaitEvent(st, e->ev_out, 0));        // the previous dose has left the staging buffer
    if ((rc = forward_impl(e, n_cp, par[0], par[1], par[2], par[3], e->s_dose.p, st))) return rc;
    CU(e, cudaEventRecord(e->ev_fwd, st));
    CU(e, cudaStreamWaitEvent(e->cs_out, e->ev_fwd, 0));
    CU(e, cudaMemcpyAsync(dose, e->s_dose.p, nvox * sizeof(float), cudaMemcpyDeviceToHost, e->cs_out));
    CU(e, cudaEventRecord(e->ev_out, e->cs_out));
    e->out_pending = true;
    return PDRT_OK;
}

int pdrt_host_wait(pdrt_engine *e)
{
    if (!e) return fail(nullptr, PDRT_EINVAL, "null engine");
    CU(e, cudaSetDevice(e->device));
    if (e->out_pending) CU(e, cudaEventSynchronize(e->ev_out));
    return PDRT_OK;
}

int pdrt_dose_host(pdrt_engine *e, int32_t n_cp, const float *leaves, const float *jaws, const float *gantry,
                   const float *mu, float *dose, void *stream)
{
    const int rc = pdrt_dose_host_async(e, n_cp, leaves, jaws, gantry, mu, dose, stream);
    return rc ? rc : pdrt_host_wait(e);
}

int pdrt_dose_backward_host(pdrt_engine *e, int32_t n_cp, const float *leaves, const float *jaws, const float *gantry,
                            const float *mu, const float *gdose, float *d_leaves, float *d_jaws, float *d_mu, void *stream)
{
    int rc = check_call(e, n_cp, { leaves, jaws, gantry, mu, gdose, d_leaves, d_jaws, d_mu });
    if (rc) return rc;
    if ((rc = host_streams(e))) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nvox = (size_t)e->P.nx * e->P.ny * e->P.nz, nl = (size_t)n_cp * 2 * e->P.Np;
    const PackOff go = pack_offsets(e, n_cp, false);
    CU(e, e->s_g.ensure(nvox)); CU(e, e->s_grad.ensure(go.total));
    if ((rc = ensure_pinned(e, &e->h_grad, &e->h_grad_n, go.total))) return rc;
    // The parameters and dL/dDose travel on the input copy stream (they need not wait for whatever still runs on this stream, e.g. the
    // forward pass of the same step); S1 / S2 wait for the parameters, the transposition of dL/dDose for the volume.
    const float *par[4];
    if ((rc = stage_params_in(e, 1, n_cp, leaves, jaws, gantry, mu, e->cs_in, par))) return rc;
    CU(e, cudaStreamWaitEvent(st, e->ev_par[1], 0));
    if (e->bwd_recorded) CU(e, cudaStreamWaitEvent(e->cs_in, e->ev_bwd, 0));  // the previous backward pass has read the staging buffer
    CU(e, cudaMemcpyAsync(e->s_g.p, gdose, nvox * sizeof(float), cudaMemcpyHostToDevice, e->cs_in));
    CU(e, cudaEventRecord(e->ev_g, e->cs_in));
    float *dg = e->s_grad.p;
    if ((rc = backward_impl(e, n_cp, par[0], par[1], par[2], par[3], e->s_g.p, dg + go.leaves, dg + go.jaws, dg + go.mu, st, e->ev_g))) return rc;
    CU(e, cudaEventRecord(e->ev_bwd, st));
    e->bwd_recorded = true;
    CU(e, cudaMemcpyAsync(e->h_grad, dg, go.total * sizeof(float), cudaMemcpyDeviceToHost, st));      // one copy; unpacked on the host
    CU(e, cudaStreamSynchronize(st));
    std::memcpy(d_leaves, e->h_grad + go.leaves, nl * sizeof(float));
    std::memcpy(d_jaws, e->h_grad + go.jaws, sizeof(float) * n_cp * 4);
    std::memcpy(d_mu, e->h_grad + go.mu, sizeof(float) * n_cp);
    return PDRT_OK;
}

int pdrt_stage_fluence(pdrt_engine *e, int32_t n_cp, const float *leaves, const float *jaws, float *phimap, void *stream)
{
    int rc = check_call(e, n_cp, { leaves, jaws, phimap });
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if ((rc = ensure_cp_scratch(e, n_cp))) return rc;
    const size_t nmap = (size_t)n_cp * e->P.Nuf * e->P.Nvf;
    CU(e, cudaMemsetAsync(e->phimap.p, 0, nmap * sizeof(float), st));     // outside the support bbox the map is zero
    set_conv_direction(e, false);
    if ((rc = run_setup(e, n_cp, leaves, jaws, nullptr, nullptr, false, st))) return rc;
    CU(e, cudaMemcpyAsync(phimap, e->phimap.p, nmap * sizeof(float), cudaMemcpyDeviceToDevice, st));
    return PDRT_OK;
}

int pdrt_stage_fan_factor(pdrt_engine *e, int32_t n_cp, const float *leaves, const float *jaws, const float *gantry, float *factor, void *stream)
{
    int rc = check_call(e, n_cp, { leaves, jaws, gantry, factor });
    if (rc) return rc;
    if (e->depth_mode != PDRT_DEPTH_FAN) return fail(e, PDRT_EINVAL, "pdrt_stage_fan_factor needs PDRT_DEPTH_FAN");
    cudaStream_t st = (cudaStream_t)stream;
    set_conv_direction(e, false);
    if ((rc = run_setup(e, n_cp, leaves, jaws, gantry, nullptr, true, st))) return rc;
    k_expand_fan<<<e->sm_count * 4, 256, 0, st>>>(e->P, e->desc.p, n_cp, e->fan_stride(), e->fan.p, factor);
    CU(e, cudaGetLastError());
    return PDRT_OK;
}

int pdrt_stage_depth(pdrt_engine *e, int32_t n_cp, const float *gantry, float *zrad, void *stream)
{
    int rc = check_call(e, n_cp, { gantry, zrad });
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if ((rc = ensure_cp_scratch(e, n_cp))) return rc;
    k_depth<<<n_cp, DEPTH_THREADS, 0, st>>>(e->P, n_cp, e->density.p, gantry, e->rho_s.p, e->Z_s.p, e->zrad.p);
    CU(e, cudaGetLastError());
    CU(e, cudaMemcpyAsync(zrad, e->zrad.p, sizeof(float) * n_cp * e->P.Nw, cudaMemcpyDeviceToDevice, st));
    return PDRT_OK;
}

int pdrt_stage_beam_dose(pdrt_engine *e, const float *leaves, const float *jaws, const float *gantry, float *db, void *stream)
{
    int rc = check_call(e, 1, { leaves, jaws, gantry, db });
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    set_conv_direction(e, false);
    if ((rc = run_setup(e, 1, leaves, jaws, gantry, nullptr, true, st))) return rc;
    CU(e, e->bufA.ensure((size_t)e->P.stride_cp));
    CU(e, e->bufB.ensure((size_t)e->P.stride_cp));
    k_scan_items<<<1, 256, 0, st>>>(e->desc.p, 0, 1, 0, e->P.Nuf, e->P.Nvf, e->tile_base.p, e->counters.p);
    CU(e, cudaGetLastError());
    k_project<<<dim3(project_blocks(e->P), 1), PROJECT_THREADS, 0, st>>>(e->P, e->desc.p, e->sbox.p, 0, 1, e->phimapT.p, e->bufB.p);
    if (e->depth_mode == PDRT_DEPTH_FAN)
        k_apply_fan<<<dim3(32, 1), 256, 0, st>>>(e->P, e->desc.p, e->sbox.p, 0, 1, e->fan_stride(), e->fan.p, e->bufB.p);
    CU(e, cudaGetLastError());
    if ((rc = launch_conv<false>(e, 0, 1, e->bufB.p, e->bufA.p, st))) return rc;
    k_expand_dense<<<e->sm_count * 4, 256, 0, st>>>(e->P, e->desc.p, e->wbox.p, 0, 0, e->bufA.p, db);
    CU(e, cudaGetLastError());
    return PDRT_OK;
}

int pdrt_stage_grad_fluence(pdrt_engine *e, int32_t n_cp, const float *leaves, const float *jaws, const float *gantry,
                            const float *gdose, float *gphimap, void *stream)
{
    int rc = check_call(e, n_cp, { leaves, jaws, gantry, gdose, gphimap });
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t nmap = (size_t)n_cp * e->P.Nuf * e->P.Nvf;
    CU(e, e->gphimap.ensure(nmap));
    CU(e, cudaMemsetAsync(e->gphimap.p, 0, nmap * sizeof(float), st));
    if ((rc = backward_to_fluence(e, n_cp, leaves, jaws, gantry, nullptr, gdose, st))) return rc;
    CU(e, cudaMemcpyAsync(gphimap, e->gphimap.p, nmap * sizeof(float), cudaMemcpyDeviceToDevice, st));
    return PDRT_OK;
}

// ---- planning loop (pdrt_plan.cuh)
float pdrt_mu_epsilon(float dose_rate_min, float delta_phi_deg, float gantry_speed_max) { return dose_rate_min * delta_phi_deg / gantry_speed_max; }

static PlanLimits plan_limits(const pdrt_limits *l) { return PlanLimits{ l->leaf_w_min, l->leaf_F, l->jaw_w_min, l->jaw_Fx, l->jaw_Fy, l->mu_eps }; }

int pdrt_validate(pdrt_engine *e, int32_t n_cp, const pdrt_limits *lim, const float *leaves, const float *jaws, const float *mu,
                  float *leaves_out, float *jaws_out, float *mu_out, void *stream)
{
    int rc = check_call(e, n_cp, { lim, leaves, jaws, mu, leaves_out, jaws_out, mu_out }, false);
    if (rc) return rc;
    const long long n = (long long)n_cp * (e->P.Np + 3);
    k_validate<false><<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(n_cp, e->P.Np, plan_limits(lim), leaves, jaws, mu, nullptr, nullptr,
                                                                                     nullptr, leaves_out, jaws_out, mu_out);
    CU(e, cudaGetLastError());
    return PDRT_OK;
}

int pdrt_validate_backward(pdrt_engine *e, int32_t n_cp, const pdrt_limits *lim, const float *leaves, const float *jaws, const float *mu,
                           const float *gl_hat, const float *gj_hat, const float *gm_hat, float *gl, float *gj, float *gm, void *stream)
{
    int rc = check_call(e, n_cp, { lim, leaves, jaws, mu, gl_hat, gj_hat, gm_hat, gl, gj, gm }, false);
    if (rc) return rc;
    const long long n = (long long)n_cp * (e->P.Np + 3);
    k_validate<true><<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(n_cp, e->P.Np, plan_limits(lim), leaves, jaws, mu, gl_hat, gj_hat,
                                                                                    gm_hat, gl, gj, gm);
    CU(e, cudaGetLastError());
    return PDRT_OK;
}

int pdrt_objective(pdrt_engine *e, const float *dose, const uint32_t *bits, int32_t n_struct, const float *lambda, const float *presc,
                   int32_t power, float *g, double *loss, void *stream)
{
    int rc = check_call(e, 1, { dose, bits, lambda, presc, g, loss }, false);
    if (rc) return rc;
    if (n_struct < 1 || n_struct > OBJ_MAX_STRUCT) return fail(e, PDRT_EINVAL, "n_struct must lie in 1..32");
    if (power != 1 && power != 2) return fail(e, PDRT_EINVAL, "power must be 1 (Eq. 10) or 2 (quadratic)");
    ObjectiveTerms T{};
    T.n = n_struct; T.power = power;
    for (int s = 0; s < n_struct; ++s) { T.lambda[s] = lambda[s]; T.presc[s] = presc[s]; }
    const int nb = e->sm_count * 8;
    CU(e, e->obj_partial.ensure(nb));
    const size_t n_vox = (size_t)e->P.nx * e->P.ny * e->P.nz;
    k_objective<<<nb, OBJ_THREADS, 0, (cudaStream_t)stream>>>(n_vox, dose, bits, T, g, e->obj_partial.p);
    CU(e, cudaGetLastError());
    k_objective_finish<<<1, 32, 0, (cudaStream_t)stream>>>(nb, e->obj_partial.p, loss);
    CU(e, cudaGetLastError());
    return PDRT_OK;
}

int pdrt_track_jaws(pdrt_engine *e, int32_t n_cp, const float *leaves, float margin, float open_gap, float *jaws, void *stream)
{
    int rc = check_call(e, n_cp, { leaves, jaws }, false);
    if (rc) return rc;
    k_track_jaws<<<(n_cp * 32 + 255) / 256, 256, 0, (cudaStream_t)stream>>>(n_cp, e->P.Np, e->T.leaf_bounds, leaves, margin, open_gap, jaws);
    CU(e, cudaGetLastError());
    return PDRT_OK;
}

int pdrt_plan_step(pdrt_engine *e, int32_t n_cp, float step_leaf, float step_mu, const float *g_leaves, const float *g_mu, float *leaves,
                   float *mu, void *stream)
{
    int rc = check_call(e, n_cp, { g_leaves, g_mu, leaves, mu }, false);
    if (rc) return rc;
    k_plan_step<<<1, STEP_THREADS, 0, (cudaStream_t)stream>>>(n_cp * 2 * e->P.Np, n_cp, step_leaf, step_mu, g_leaves, g_mu, leaves, mu);
    CU(e, cudaGetLastError());
    return PDRT_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// pdrt_objective_noalloc — pdrt_objective (Eq. 10 / quadratic) for callers that cannot allocate device
// memory (stream capture, serving loops, harnesses that forbid it).  Its scratch — the block partials of the loss and the
// ticket that elects the block which adds them up — lives in a file-scope __device__ array of fixed size; the call makes
// no cudaMalloc / cudaFree and uses no engine scratch.
//
// In host code `g_noalloc_scratch` is a host-side stand-in for the symbol, NOT a device address: the address is resolved
// with cudaGetSymbolAddress once per device (that device current) and handed to the kernel as a plain pointer.
namespace {

constexpr int NOALLOC_TILE = OBJ_THREADS * 16;                                  // voxels per block: fixed, so that the
                                                                                // summation order does not depend on the GPU
constexpr int NOALLOC_MAX_PARTIALS = PDRT_NOALLOC_MAX_VOXELS / NOALLOC_TILE;    // 8192 block partials
constexpr int NOALLOC_HEADER = 32;                                              // doubles in front of the partials (256 bytes):
                                                                                // the ticket (unsigned) sits in the first 4 bytes
static_assert((long long)NOALLOC_MAX_PARTIALS * NOALLOC_TILE == PDRT_NOALLOC_MAX_VOXELS, "the maximum is a whole number of tiles");

}  // namespace

// 64.25 KiB per GPU that loads the library, held until the process exits.  Shared by every call on that GPU.
static __device__ __align__(256) double g_noalloc_scratch[NOALLOC_HEADER + NOALLOC_MAX_PARTIALS];

namespace {

// k_objective with a fixed tile of voxels per block and the final sum folded in: every block writes its float64 partial to
// scratch[NOALLOC_HEADER + block]; the block that draws the last ticket adds the partials in index order (thread t takes
// t, t + 256, ...; then a fixed tree) and writes the loss.  The per-voxel arithmetic and the order of the structures are
// those of k_objective, so dL/dDose is bit-identical; the loss differs from k_objective's by float64 rounding order only.
// The ticket must be zero at launch (the entry point clears it on the stream); the partials need no clearing.
__global__ void __launch_bounds__(OBJ_THREADS)
k_objective_noalloc(size_t n_vox, const float *__restrict__ dose, const unsigned *__restrict__ bits, ObjectiveTerms T, float *__restrict__ g,
                    double *scratch, double *__restrict__ loss)
{
    __shared__ double red[OBJ_THREADS];
    __shared__ bool last;
    unsigned *ticket = reinterpret_cast<unsigned *>(scratch);
    double *partial = scratch + NOALLOC_HEADER;
    const size_t base = (size_t)blockIdx.x * NOALLOC_TILE;
    double L = 0.0;
#pragma unroll 4
    for (int q = 0; q < NOALLOC_TILE / OBJ_THREADS; ++q) {
        const size_t x = base + (size_t)q * OBJ_THREADS + threadIdx.x;
        if (x >= n_vox) break;
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
    red[threadIdx.x] = L;
    __syncthreads();
    for (int o = OBJ_THREADS / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        partial[blockIdx.x] = red[0];
        __threadfence();                                     // the partial is visible before the ticket is drawn
        last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    const volatile double *pv = partial;                     // written by other blocks during this launch: no cached reads
    double s = 0.0;
    for (unsigned b = threadIdx.x; b < gridDim.x; b += OBJ_THREADS) s += pv[b];
    red[threadIdx.x] = s;
    __syncthreads();
    for (int o = OBJ_THREADS / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) red[threadIdx.x] += red[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) { *loss = red[0]; *ticket = 0u; }
}

constexpr int NOALLOC_MAX_DEVICES = 64;
double *g_noalloc_addr[NOALLOC_MAX_DEVICES] = {};            // device address of g_noalloc_scratch, per device ordinal
std::mutex g_noalloc_mutex;

// Device address of the scratch array on the engine's device (current: check_call has set it).  Resolved once per device.
int noalloc_scratch(pdrt_engine *e, double **out)
{
    if (e->device < 0 || e->device >= NOALLOC_MAX_DEVICES) return fail(e, PDRT_EINVAL, "pdrt_objective_noalloc: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_noalloc_mutex);
    if (!g_noalloc_addr[e->device]) {
        void *p = nullptr;
        CU(e, cudaGetSymbolAddress(&p, g_noalloc_scratch));
        if (!p) return fail(e, PDRT_ECUDA, "pdrt_objective_noalloc: cudaGetSymbolAddress returned a null address");
        g_noalloc_addr[e->device] = static_cast<double *>(p);
    }
    *out = g_noalloc_addr[e->device];
    return PDRT_OK;
}

}  // namespace

extern "C" {

int pdrt_objective_noalloc(pdrt_engine *e, const float *dose, const uint32_t *bits, int32_t n_struct, const float *lambda, const float *presc,
                           int32_t power, float *g, double *loss, void *stream)
{
    int rc = check_call(e, 1, { dose, bits, lambda, presc, g, loss }, false);
    if (rc) return rc;
    if (n_struct < 1 || n_struct > OBJ_MAX_STRUCT) return fail(e, PDRT_EINVAL, "n_struct must lie in 1..32");
    if (power != 1 && power != 2) return fail(e, PDRT_EINVAL, "power must be 1 (Eq. 10) or 2 (quadratic)");
    const size_t n_vox = (size_t)e->P.nx * e->P.ny * e->P.nz;
    if (n_vox > (size_t)PDRT_NOALLOC_MAX_VOXELS)
        return fail(e, PDRT_EINVAL, "pdrt_objective_noalloc: the dose grid has " + std::to_string(n_vox) + " voxels, the static scratch serves at most " +
                                        std::to_string((long long)PDRT_NOALLOC_MAX_VOXELS) + " (PDRT_NOALLOC_MAX_VOXELS); use pdrt_objective");
    ObjectiveTerms T{};
    T.n = n_struct; T.power = power;
    for (int s = 0; s < n_struct; ++s) { T.lambda[s] = lambda[s]; T.presc[s] = presc[s]; }
    double *scratch = nullptr;
    if ((rc = noalloc_scratch(e, &scratch))) return rc;
    const unsigned nb = (unsigned)((n_vox + NOALLOC_TILE - 1) / NOALLOC_TILE);
    CU(e, cudaMemsetAsync(scratch, 0, NOALLOC_HEADER * sizeof(double), (cudaStream_t)stream));      // the ticket starts at zero whatever the last call left
    k_objective_noalloc<<<nb, OBJ_THREADS, 0, (cudaStream_t)stream>>>(n_vox, dose, bits, T, g, scratch, loss);
    CU(e, cudaGetLastError());
    return PDRT_OK;
}

}  // extern "C"
