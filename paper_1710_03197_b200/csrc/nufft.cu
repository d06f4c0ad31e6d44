// nufft.cu -- the C-ABI library of the B200-native NUFFT hot path (include/nufft.h): plan creation (host, float64),
// kernel launches for A = V F S, A^H = S^H F^H V^H, A^H A, the multi-coil operator and the CG / L1TV-OLS drivers.
// Product path: no CPU fallback, no cuFFT, nothing from oracle/.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/nufft.h"
#include "common.cuh"
#include "fft.cuh"
#include "plan.hpp"
#include "solver.cuh"
#include "spread_interp.cuh"
#include "batch_il.cuh"
#include "win3d.cuh"

using namespace nufft;

static thread_local int g_last_cuda_error = 0;

#define CU_TRY(expr)                                        \
    do {                                                    \
        cudaError_t e__ = (expr);                           \
        if (e__ != cudaSuccess) {                           \
            g_last_cuda_error = (int)e__;                   \
            (void)cudaGetLastError();                       \
            return NUFFT_ECUDA;                             \
        }                                                   \
    } while (0)
#define NU_TRY(expr)                 \
    do {                             \
        int r__ = (expr);            \
        if (r__ != NUFFT_OK) return r__; \
    } while (0)

// identity of the captured CG iteration (operator configuration and every pointer baked into the graph)
struct CgGraphKey {
    bool coils, tv;
    float mu, lam;
    bool toep;
    const void *x, *r, *pv, *Ap, *hist, *stream;
};

struct nufft_plan_s {
    int d = 0;
    int device = -1;                // the CUDA device the plan was created on (every call must run with it current)
    int N[3] = {1, 1, 1}, K[3] = {1, 1, 1};
    int64_t M = 0, nimg = 0, cells = 0;
    int max_batch = 1;
    nufft_opts opts{};
    int J = kJ;                     // kernel width (uniform over the axes); J != kJ runs the direct V / atomic V^H kernels
    KernelPoly poly{};
    KernelPolyG polyg{};            // J != kJ
    bool generic_j = false;         // J != kJ, or opts.interp_mode == 2 (the same kernels at J = kJ, for cross-checks)
    bool generic_sigma = false;     // Kd != 2 Nd: unpruned FFT + separate pad / crop kernels, planar, direct or tiled V / V^H
    bool minmax = false;            // opts.kernel == 1: min-max interpolator (reading R25); only the weight polynomials
    host::MinMaxKernel mm[3];       //   and the float64 V^H table differ from the Kaiser-Bessel plan (one per axis: N_a)
    double poly_err = 0.0;
    // device plan data
    float* d_scale[3] = {nullptr, nullptr, nullptr};
    float2* d_tw[3] = {nullptr, nullptr, nullptr};
    uint32_t* d_kpack = nullptr;
    float* d_delta = nullptr;
    int32_t* d_perm = nullptr;
    // workspace
    float2* d_grid = nullptr;       // [max_batch][cells]
    float2* d_ywork = nullptr;      // [max_batch][M]     (selfadjoint intermediate)
    float2* d_imgwork = nullptr;    // [max_batch][nimg]  (per-coil images of the multi-coil adjoint), lazy
    float2* d_solver = nullptr;     // solver vectors, lazy
    int64_t solver_vecs = 0;
    CgScalars* d_scal = nullptr;
    double* d_hist = nullptr;
    int hist_cap = 0;
    // coils (borrowed)
    int ncoil = 0;
    const float2* d_coils = nullptr;
    // tiles and V^H work items
    int tile[3] = {1, 1, 1}, ntile[3] = {1, 1, 1};
    TileGeom tg{};
    WorkItem* d_items = nullptr;
    int32_t* d_tile_item_start = nullptr;
    int n_items = 0;
    float2* d_slabs = nullptr;      // deterministic mode: [max_batch][n_items][tile_cells], lazy
    int64_t n_tiles = 0, n_work = 0, max_tile_samples = 0;
    int64_t tile_hist[NUFFT_TILE_HIST_BUCKETS] = {0};
    float* d_w3rec = nullptr;       // coef_mode = 1, win3d: per-sample records [M][28] (padded weights, window key, caller index)
    float* d_il_wv = nullptr;       // coef_mode = 1, interleaved V: padded weights [M][16] in V order / caller order
    float* d_il_wv_c = nullptr;
    bool win3d = false;             // 3-D, J = 6, default tile: samples pencil-sorted inside tiles, register-window V / V^H (win3d.cuh)
    int64_t bytes_plan = 0, bytes_work = 0;
    int64_t launches = 0;
    // batch-interleaved 2-D path (batch_il.cuh): cell-sorted plan data, V^H weight table, row pointers, work items
    bool il_ok = false;
    int il_min_batch = 12;
    int batch_pad = 1;              // max_batch rounded up to whole groups of 32 when il_ok
    uint32_t* d_il_kpack = nullptr;
    float* d_il_delta = nullptr;
    int32_t* d_il_pos = nullptr;     // caller sample -> V^H-order position (the order of y_il)
    float* d_il_wtab = nullptr;
    int32_t* d_il_rowptr = nullptr;
    int32_t* d_il_v2h = nullptr;     // V-order position -> V^H-order position
    uint32_t* d_il_gbase = nullptr;      // window-group base cell per sample, V order / caller order (interp_il_win_kernel)
    uint32_t* d_il_gbase_c = nullptr;
    uint32_t* d_il_kpack_c = nullptr;    // caller-order copies for trajectory-coherent plans (il_coherent)
    float* d_il_delta_c = nullptr;
    bool il_coherent = false;
    IlItem* d_il_items = nullptr;
    int n_il_items = 0;
    uint32_t* d_il_kpack_t = nullptr;    // tile order of interp_il_tile_kernel
    float* d_il_delta_t = nullptr;
    uint32_t* d_il_gbase_t = nullptr;
    float* d_il_wv_t = nullptr;
    int32_t* d_il_t2h = nullptr;
    IlTileItem* d_il_titems = nullptr;
    int n_il_titems = 0;
    float2* noalloc_grid = nullptr;     // device address of g_noalloc_grid on the plan's device (nufft_adjoint_noalloc), or null
    float2* d_yil = nullptr;        // [groups][M][32] sorted, interleaved samples (adjoint input), lazy
    // "next" rows: density compensation and Toeplitz A^H A
    std::vector<double> om_host;    // copy of the trajectory (the Toeplitz build plans a second, 2N transform)
    float* d_ones = nullptr;        // unit scaling vector (max N), used instead of d_scale by the Toeplitz passes
    float2* d_that = nullptr;       // Toeplitz spectrum T^ on the K grid, planar [K0][K1]([K2])
    bool toep_on = false;           // solvers and selfadjoint calls use the Toeplitz operator
    bool unit_scale = false;        // transient: FFT row passes use d_ones
    bool inv_scale = false;         // transient: FFT row passes use d_sinv (1 / (s K)): x = S^-1 F^-1 k of eq. (10)
    float* d_sinv[3] = {nullptr, nullptr, nullptr};
    float2* d_kspace = nullptr;     // 5 grid-sized vectors of the k-space CG, lazy
    const float2* cur_mult = nullptr;   // transient: the first adjoint column pass multiplies by this spectrum
    float2* d_dcf_img = nullptr;
    float2* d_dcf_t = nullptr;
    struct OpGraph { int kind, batch; const void* in; void* out; void* stream; cudaGraphExec_t exec; int launches; };
    std::vector<OpGraph> op_graphs;         // replayable transform calls (opts.use_graphs)
    bool op_warm[3][2] = {{false, false}, {false, false}, {false, false}};
    cudaGraphExec_t cg_graph = nullptr;     // one CG iteration (opts.use_graphs)
    CgGraphKey cg_key{};
    int cg_iter_launches = 0;
    // host-buffer pipeline (nufft_*_host): copy streams, events, double-buffered device staging, lazy
    bool hp_ready = false;
    bool hp_input_ready = false;    // nufft_host_input_ready
    bool hp_used[2] = {false, false};
    int hp_chunk = 1;
    cudaStream_t hp_h2d = nullptr, hp_d2h = nullptr;
    cudaEvent_t hp_in[2] = {nullptr, nullptr}, hp_cmp[2] = {nullptr, nullptr}, hp_out[2] = {nullptr, nullptr}, hp_start = nullptr;
    float2* hp_din[2] = {nullptr, nullptr};
    float2* hp_dout[2] = {nullptr, nullptr};
    // optional per-kernel event timing (nufft_profile_*)
    bool prof_on = false;
    struct ProfRec { int label; cudaEvent_t a, b; };
    std::vector<ProfRec> prof;
    std::vector<const char*> prof_labels;
    std::vector<double> prof_ms;
    std::vector<int64_t> prof_n;
};

// Brackets the launches issued during its lifetime with a pair of events when profiling is enabled.
struct ProfScope {
    nufft_plan_t p;
    cudaStream_t st;
    int idx = -1;
    ProfScope(nufft_plan_t p_, const char* label, cudaStream_t st_) : p(p_), st(st_) {
        if (!p->prof_on) return;
        int li = -1;
        for (size_t i = 0; i < p->prof_labels.size(); ++i)
            if (p->prof_labels[i] == label || std::strcmp(p->prof_labels[i], label) == 0) { li = (int)i; break; }
        if (li < 0) { li = (int)p->prof_labels.size(); p->prof_labels.push_back(label); p->prof_ms.push_back(0.0); p->prof_n.push_back(0); }
        nufft_plan_s::ProfRec r{li, nullptr, nullptr};
        if (cudaEventCreate(&r.a) != cudaSuccess || cudaEventCreate(&r.b) != cudaSuccess) return;
        cudaEventRecord(r.a, st);
        idx = (int)p->prof.size();
        p->prof.push_back(r);
    }
    ~ProfScope() {
        if (idx >= 0) cudaEventRecord(p->prof[idx].b, st);
    }
};

static int dev_alloc(void** dptr, size_t bytes, int64_t* acct);
static bool wrong_device(nufft_plan_t p);

// ------------------------------------------------------------------------------------------------------------
// kernel configuration (dynamic shared memory opt-in), once per process
// ------------------------------------------------------------------------------------------------------------
template <int K> static size_t smem_rows() { return (size_t)Rad<K>::LC * FftGeom<K>::PITCH_C * sizeof(float2); }
template <int K> static size_t smem_cols() { return (size_t)Rad<K>::TS * FftGeom<K>::SIZE_S * sizeof(float2); }

template <int K> static cudaError_t configure_fft() {
    cudaError_t e;
    e = cudaFuncSetAttribute(fft_rows_fwd_kernel<K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_rows<K>());
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(fft_rows_adj_kernel<K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_rows<K>());
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(fft_cols_kernel<K, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_cols<K>());
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(fft_cols_kernel<K, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_cols<K>());
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(fft_il_rows_fwd_kernel<K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_cols<K>());
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(fft_il_rows_adj_kernel<K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_cols<K>());
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(fft_il_rows_adj_coilsum_kernel<K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_cols<K>());
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(fft_cols_kernel<K, true, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_cols<K>());
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(fft_cols_kernel<K, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_cols<K>());
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(fft_rows_full_kernel<K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_rows<K>());
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(fft_rows_pad_kernel<K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_rows<K>());
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(fft_rows_crop_kernel<K>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_rows<K>());
    return e;
}

static cudaError_t configure_all() {
    cudaError_t e;
    if ((e = configure_fft<32>()) != cudaSuccess) return e;
    if ((e = configure_fft<64>()) != cudaSuccess) return e;
    if ((e = configure_fft<128>()) != cudaSuccess) return e;
    if ((e = configure_fft<256>()) != cudaSuccess) return e;
    if ((e = configure_fft<512>()) != cudaSuccess) return e;
    if ((e = configure_fft<1024>()) != cudaSuccess) return e;
    const int big = 200 * 1024;
    if ((e = cudaFuncSetAttribute(gridding_tiled_2d_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, big)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(interp_tiled_2d_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, big)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(gridding_tiled_2d_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, big)) != cudaSuccess) return e;
#define NU_TILED_J_CFG(JJ) if ((e = cudaFuncSetAttribute(gridding_tiled_2d_j_kernel<JJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, big)) != cudaSuccess) return e;
    NU_TILED_J_CFG(2) NU_TILED_J_CFG(3) NU_TILED_J_CFG(4) NU_TILED_J_CFG(5) NU_TILED_J_CFG(6) NU_TILED_J_CFG(7) NU_TILED_J_CFG(8)
#undef NU_TILED_J_CFG
    if ((e = cudaFuncSetAttribute(gridding_tiled_3d_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, big)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(interp_tiled_3d_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kInterp3dSmem)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(gridding_il_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, GridStage<1>::BYTES)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(interp_il_tile_kernel<kItT, kItWarps, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, IlTile<kItT, kItWarps>::SMEM)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(gridding_il_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, GridStage<2>::BYTES)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(gridding_tiled_3d_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, big)) != cudaSuccess) return e;
#define NU_W3_CFG(NW)                                                                                                                   \
    if ((e = cudaFuncSetAttribute(interp_win_3d_kernel<NW, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, win3d_smem(NW))) != cudaSuccess) return e;   \
    if ((e = cudaFuncSetAttribute(interp_win_3d_kernel<NW, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, win3d_smem(NW))) != cudaSuccess) return e;   \
    if ((e = cudaFuncSetAttribute(gridding_win_3d_kernel<NW, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, win3d_smem(NW))) != cudaSuccess) return e; \
    if ((e = cudaFuncSetAttribute(gridding_win_3d_kernel<NW, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, win3d_smem(NW))) != cudaSuccess) return e;
    NU_W3_CFG(kW3InterpWarps) NU_W3_CFG(kW3GridWarps)
#undef NU_W3_CFG
    return cudaSuccess;
}

// ------------------------------------------------------------------------------------------------------------
// FFT pass launchers
// ------------------------------------------------------------------------------------------------------------
// launch with programmatic stream serialization (see pdl_enter in common.cuh).  Measured (cfg2 batch 64): it shortens the
// forward chain of the interleaved path (0.1905 -> 0.1827 ms) but LENGTHENS its adjoint chain (0.2059 -> 0.2205 ms: the
// early-resident CTAs of the next kernel take shared memory from the tail of gridding_il), so the interleaved adjoint runners
// switch it off (PdlOff); the planar path keeps it in both directions (batch-1 adjoint 34.8 -> 27.7 us).
static thread_local bool t_pdl = true;
struct PdlOff {
    bool prev;
    PdlOff() : prev(t_pdl) { t_pdl = false; }
    ~PdlOff() { t_pdl = prev; }
};
template <class... KArgs, class... Args>
static void launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = t_pdl ? 1 : 0;
    (void)cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

template <int K> static void launch_rows(bool adj, const RowPassParams& p, cudaStream_t st) {
    constexpr int threads = FftGeom<K>::TPL * Rad<K>::LC;
    const int blocks = (p.nlines + Rad<K>::LC - 1) / Rad<K>::LC;
    if (adj) launch_pdl(fft_rows_adj_kernel<K>, dim3(blocks), dim3(threads), smem_rows<K>(), st, p);
    else     launch_pdl(fft_rows_fwd_kernel<K>, dim3(blocks), dim3(threads), smem_rows<K>(), st, p);
}
template <int K> static void launch_cols(bool adj, const ColPassParams& p, cudaStream_t st) {
    constexpr int threads = FftGeom<K>::TPL * Rad<K>::TS;
    if (adj && p.mult) launch_pdl(fft_cols_kernel<K, true, false, true>, dim3(p.ngroups), dim3(threads), smem_cols<K>(), st, p);
    else if (adj) launch_pdl(fft_cols_kernel<K, true>, dim3(p.ngroups), dim3(threads), smem_cols<K>(), st, p);
    else     launch_pdl(fft_cols_kernel<K, false>, dim3(p.ngroups), dim3(threads), smem_cols<K>(), st, p);
}
static int tile_T(int K) {
    switch (K) {
        case 32: return Rad<32>::TS; case 64: return Rad<64>::TS; case 128: return Rad<128>::TS;
        case 256: return Rad<256>::TS; case 512: return Rad<512>::TS; case 1024: return Rad<1024>::TS;
    }
    return 0;
}
static int dispatch_rows(int K, bool adj, const RowPassParams& p, cudaStream_t st) {
    switch (K) {
        case 32: launch_rows<32>(adj, p, st); break;
        case 64: launch_rows<64>(adj, p, st); break;
        case 128: launch_rows<128>(adj, p, st); break;
        case 256: launch_rows<256>(adj, p, st); break;
        case 512: launch_rows<512>(adj, p, st); break;
        case 1024: launch_rows<1024>(adj, p, st); break;
        default: return NUFFT_EINVAL;
    }
    CU_TRY(cudaGetLastError());
    return NUFFT_OK;
}
static int dispatch_cols(int K, bool adj, const ColPassParams& p, cudaStream_t st) {
    switch (K) {
        case 32: launch_cols<32>(adj, p, st); break;
        case 64: launch_cols<64>(adj, p, st); break;
        case 128: launch_cols<128>(adj, p, st); break;
        case 256: launch_cols<256>(adj, p, st); break;
        case 512: launch_cols<512>(adj, p, st); break;
        case 1024: launch_cols<1024>(adj, p, st); break;
        default: return NUFFT_EINVAL;
    }
    CU_TRY(cudaGetLastError());
    return NUFFT_OK;
}

static RowPassParams row_params(nufft_plan_t p, int batch, const float2* img_in, float2* img_out, float2* grid,
                                const float2* coil, bool same_image) {
    RowPassParams r{};
    r.img_in = img_in; r.img_out = img_out; r.grid = grid; r.coil = coil;
    const int d = p->d;
    auto sc = [&](int a) -> const float* { return p->unit_scale ? p->d_ones : (p->inv_scale ? p->d_sinv[a] : p->d_scale[a]); };
    r.s_line = sc(d - 1);
    r.tw = p->d_tw[d - 1];
    if (d == 1) {          // one line per image: no outer axes
        r.s_outer0 = p->d_ones; r.s_outer1 = nullptr;
        r.n_outer0 = 1; r.n_outer1 = 1; r.k_outer0 = 1; r.k_outer1 = 1;
    } else if (d == 2) {
        r.s_outer0 = sc(0); r.s_outer1 = nullptr;
        r.n_outer0 = p->N[0]; r.n_outer1 = 1; r.k_outer0 = p->K[0]; r.k_outer1 = 1;
    } else {
        r.s_outer0 = sc(0); r.s_outer1 = sc(1);
        r.n_outer0 = p->N[0]; r.n_outer1 = p->N[1]; r.k_outer0 = p->K[0]; r.k_outer1 = p->K[1];
    }
    r.nlines = batch * r.n_outer0 * r.n_outer1;
    r.img_batch_stride_is_zero = same_image ? 1 : 0;
    return r;
}

static int fft_full_inplace(nufft_plan_t p, float2* data, cudaStream_t st, int batch = 1, bool do_rows = true);
static PadGeom pad_geom(nufft_plan_t p) {
    PadGeom g{};
    g.d = p->d;
    for (int a = 0; a < 3; ++a) {
        g.N[a] = p->N[a]; g.K[a] = p->K[a];
        g.s[a] = p->unit_scale ? p->d_ones : (p->inv_scale ? p->d_sinv[a] : p->d_scale[a]);
    }
    return g;
}
static int ew_blocks(int64_t n);

// sigma != 2: contiguous-axis pass with S + zero-pad (forward) / crop + S^H (adjoint) fused (fft.cuh)
template <int K> static void launch_rows_sigma(bool adj, const SigmaRowParams& sp, cudaStream_t st) {
    constexpr int threads = FftGeom<K>::TPL * Rad<K>::LC;
    const int blocks = (sp.nlines + Rad<K>::LC - 1) / Rad<K>::LC;
    if (adj) launch_pdl(fft_rows_crop_kernel<K>, dim3(blocks), dim3(threads), smem_rows<K>(), st, sp);
    else     launch_pdl(fft_rows_pad_kernel<K>, dim3(blocks), dim3(threads), smem_rows<K>(), st, sp);
}
static int dispatch_rows_sigma(nufft_plan_t p, bool adj, int batch, const float2* x_in, float2* x_out, float2* grid,
                               const float2* coil, bool same_image, cudaStream_t st) {
    SigmaRowParams sp{};
    sp.g = pad_geom(p);
    sp.img_in = x_in; sp.img_out = x_out; sp.grid = grid; sp.coil = coil;
    sp.tw = p->d_tw[p->d - 1];
    sp.cells = p->cells; sp.nimg = p->nimg; sp.same_image = same_image ? 1 : 0;
    int64_t lines = batch;
    for (int a = 0; a + 1 < p->d; ++a) lines *= adj ? p->N[a] : p->K[a];
    sp.nlines = (int)lines;
    switch (p->K[p->d - 1]) {
        case 32: launch_rows_sigma<32>(adj, sp, st); break;
        case 64: launch_rows_sigma<64>(adj, sp, st); break;
        case 128: launch_rows_sigma<128>(adj, sp, st); break;
        case 256: launch_rows_sigma<256>(adj, sp, st); break;
        case 512: launch_rows_sigma<512>(adj, sp, st); break;
        case 1024: launch_rows_sigma<1024>(adj, sp, st); break;
        default: return NUFFT_EINVAL;
    }
    CU_TRY(cudaGetLastError());
    p->launches++;
    return NUFFT_OK;
}

// a1 + a2: grid = F S x  (coil != nullptr: grid_b = F S (c_b . x))
static int run_scale_fft(nufft_plan_t p, int batch, const float2* x, float2* grid, const float2* coil,
                         bool same_image, cudaStream_t st) {
    const int d = p->d;
    if (p->generic_sigma) {      // sigma != 2: S + zero-pad fused into the unpruned contiguous-axis pass, then the strided passes
        { ProfScope ps(p, "fft_rows_fwd", st); NU_TRY(dispatch_rows_sigma(p, false, batch, x, nullptr, grid, coil, same_image, st)); }
        if (d == 1) return NUFFT_OK;
        ProfScope ps(p, "fft_full_fwd", st);
        return fft_full_inplace(p, grid, st, batch, false);
    }
    RowPassParams r = row_params(p, batch, x, nullptr, grid, coil, same_image);
    { ProfScope ps(p, "fft_rows_fwd", st); NU_TRY(dispatch_rows(p->K[d - 1], false, r, st)); }
    p->launches++;
    if (d == 1) return NUFFT_OK;
    if (d == 2) {
        ColPassParams c{};
        c.grid = grid; c.tw = p->d_tw[0];
        c.batch_stride = p->cells; c.outer_stride = 0; c.line_stride = p->K[1];
        c.n_outer = 1; c.k_outer = 0; c.inner = p->K[1];
        c.ngroups = batch * (c.inner / tile_T(p->K[0]));
        { ProfScope ps(p, "fft_cols_fwd", st); NU_TRY(dispatch_cols(p->K[0], false, c, st)); }
        p->launches++;
    } else {
        ColPassParams c{};
        c.grid = grid; c.tw = p->d_tw[1];
        c.batch_stride = p->cells; c.outer_stride = (int64_t)p->K[1] * p->K[2]; c.line_stride = p->K[2];
        c.n_outer = p->N[0]; c.k_outer = p->K[0]; c.inner = p->K[2];
        c.ngroups = batch * c.n_outer * (c.inner / tile_T(p->K[1]));
        { ProfScope ps(p, "fft_cols_fwd_axis1", st); NU_TRY(dispatch_cols(p->K[1], false, c, st)); }
        ColPassParams c0{};
        c0.grid = grid; c0.tw = p->d_tw[0];
        c0.batch_stride = p->cells; c0.outer_stride = 0; c0.line_stride = (int64_t)p->K[1] * p->K[2];
        c0.n_outer = 1; c0.k_outer = 0; c0.inner = p->K[1] * p->K[2];
        c0.ngroups = batch * (c0.inner / tile_T(p->K[0]));
        { ProfScope ps(p, "fft_cols_fwd_axis0", st); NU_TRY(dispatch_cols(p->K[0], false, c0, st)); }
        p->launches += 2;
    }
    return NUFFT_OK;
}

// a5 + a6: x = S^H F^H grid  (grid destroyed; coil != nullptr: x_b = conj(c_b) . S^H F^H grid_b)
static int run_fft_scale(nufft_plan_t p, int batch, float2* grid, float2* x, const float2* coil, cudaStream_t st) {
    const int d = p->d;
    if (p->generic_sigma) {      // sigma != 2: unpruned strided passes, then the contiguous-axis pass on the kept lines only with
        if (d > 1) { ProfScope ps(p, "fft_full_adj", st); NU_TRY(fft_full_inplace(p, grid, st, batch, false)); }   // crop (reversed index = F^H) + S^H fused
        ProfScope ps(p, "fft_rows_adj", st);
        return dispatch_rows_sigma(p, true, batch, nullptr, x, grid, coil, false, st);
    }
    if (d == 1) {
        // the Toeplitz spectrum multiply normally rides on the first adjoint column pass; 1-D has none
        if (p->cur_mult) {
            spectrum_mul_kernel<<<(int)std::max<int64_t>(1, std::min<int64_t>((p->cells * batch + 255) / 256, 148 * 8)), 256, 0, st>>>(grid, p->cur_mult, p->cells, batch);
            CU_TRY(cudaGetLastError());
            p->launches++;
        }
    } else if (d == 2) {
        ColPassParams c{};
        c.grid = grid; c.tw = p->d_tw[0];
        c.batch_stride = p->cells; c.outer_stride = 0; c.line_stride = p->K[1];
        c.n_outer = 1; c.k_outer = 0; c.inner = p->K[1];
        c.ngroups = batch * (c.inner / tile_T(p->K[0]));
        c.mult = p->cur_mult; c.mult_shift = 0;
        { ProfScope ps(p, "fft_cols_adj", st); NU_TRY(dispatch_cols(p->K[0], true, c, st)); }
        p->launches++;
    } else {
        ColPassParams c0{};
        c0.grid = grid; c0.tw = p->d_tw[0];
        c0.batch_stride = p->cells; c0.outer_stride = 0; c0.line_stride = (int64_t)p->K[1] * p->K[2];
        c0.n_outer = 1; c0.k_outer = 0; c0.inner = p->K[1] * p->K[2];
        c0.ngroups = batch * (c0.inner / tile_T(p->K[0]));
        c0.mult = p->cur_mult; c0.mult_shift = 0;
        { ProfScope ps(p, "fft_cols_adj_axis0", st); NU_TRY(dispatch_cols(p->K[0], true, c0, st)); }
        ColPassParams c{};
        c.grid = grid; c.tw = p->d_tw[1];
        c.batch_stride = p->cells; c.outer_stride = (int64_t)p->K[1] * p->K[2]; c.line_stride = p->K[2];
        c.n_outer = p->N[0]; c.k_outer = p->K[0]; c.inner = p->K[2];
        c.ngroups = batch * c.n_outer * (c.inner / tile_T(p->K[1]));
        { ProfScope ps(p, "fft_cols_adj_axis1", st); NU_TRY(dispatch_cols(p->K[1], true, c, st)); }
        p->launches += 2;
    }
    RowPassParams r = row_params(p, batch, nullptr, x, grid, coil, false);
    { ProfScope ps(p, "fft_rows_adj", st); NU_TRY(dispatch_rows(p->K[d - 1], true, r, st)); }
    p->launches++;
    return NUFFT_OK;
}

static GridGeom grid_geom(nufft_plan_t p) {
    GridGeom g{};
    g.K[0] = p->K[0]; g.K[1] = p->K[1]; g.K[2] = p->K[2];
    g.cells = p->cells; g.M = p->M;
    return g;
}
static SampleData sample_data(nufft_plan_t p) {
    SampleData s{};
    s.kpack = p->d_kpack; s.delta = p->d_delta; s.perm = p->d_perm;
    return s;
}

// Tensor map of a planar 3-D grid [batch][K0][K1][K2] complex64 seen as float32 [batch][K0][K1][2 K2], box = one padded
// tile (win3d.cuh).  cuTensorMapEncodeTiled is a host-only driver entry point (no context work), fetched through the
// runtime so that libcuda is not a link dependency.  Returns false when the driver cannot provide it: the kernels then
// stage and flush tiles row by row.
typedef CUresult (*tmap_encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                   const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                   CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static tmap_encode_fn tmap_encoder() {
    static tmap_encode_fn fn = []() -> tmap_encode_fn {
        void* f = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess) { (void)cudaGetLastError(); return nullptr; }
        return (tmap_encode_fn)f;
    }();
    return fn;
}
static bool tile_tensor_map(nufft_plan_t p, int batch, const float2* grid, CUtensorMap* tm) {
    std::memset(tm, 0, sizeof(*tm));
    tmap_encode_fn enc = tmap_encoder();
    if (!enc) return false;
    const cuuint32_t est[4] = {1, 1, 1, 1};
    if (p->d == 3) {
        const cuuint64_t gdim[4] = {(cuuint64_t)2 * p->K[2], (cuuint64_t)p->K[1], (cuuint64_t)p->K[0], (cuuint64_t)batch};
        const cuuint64_t gstr[3] = {(cuuint64_t)p->K[2] * 8, (cuuint64_t)p->K[1] * p->K[2] * 8, (cuuint64_t)p->cells * 8};
        const cuuint32_t box[4] = {2 * k3Pitch, k3P1, k3P0, 1};
        return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (void*)grid, gdim, gstr, box, est, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
    }
    if (p->d == 2) {      // planar 2-D grid [batch][K0][K1] as float32 [batch][K0][2 K1]; box = one padded V / V^H tile
        if (2 * p->tg.pitch > 256 || p->tg.P[0] > 256) return false;
        const cuuint64_t gdim[3] = {(cuuint64_t)2 * p->K[1], (cuuint64_t)p->K[0], (cuuint64_t)batch};
        const cuuint64_t gstr[2] = {(cuuint64_t)p->K[1] * 8, (cuuint64_t)p->cells * 8};
        const cuuint32_t box[3] = {(cuuint32_t)(2 * p->tg.pitch), (cuuint32_t)p->tg.P[0], 1};
        return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void*)grid, gdim, gstr, box, est, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
    }
    return false;
}

// Widths other than kJ: direct V and atomic V^H, one instantiation per (d, J)
#define NU_J_CASES(KERNEL, D, ...)                                                             \
    switch (p->J) {                                                                            \
    case 2: KERNEL<D, 2, KernelPolyG><<<blocks, 128, 0, st>>>(__VA_ARGS__); break;             \
    case 3: KERNEL<D, 3, KernelPolyG><<<blocks, 128, 0, st>>>(__VA_ARGS__); break;             \
    case 4: KERNEL<D, 4, KernelPolyG><<<blocks, 128, 0, st>>>(__VA_ARGS__); break;             \
    case 5: KERNEL<D, 5, KernelPolyG><<<blocks, 128, 0, st>>>(__VA_ARGS__); break;             \
    case 6: KERNEL<D, 6, KernelPolyG><<<blocks, 128, 0, st>>>(__VA_ARGS__); break;             \
    case 7: KERNEL<D, 7, KernelPolyG><<<blocks, 128, 0, st>>>(__VA_ARGS__); break;             \
    case 8: KERNEL<D, 8, KernelPolyG><<<blocks, 128, 0, st>>>(__VA_ARGS__); break;             \
    default: return NUFFT_EINVAL;                                                              \
    }
#define NU_DJ_CASES(KERNEL, ...)                                                               \
    if (p->d == 1) { NU_J_CASES(KERNEL, 1, __VA_ARGS__) }                                      \
    else if (p->d == 2) { NU_J_CASES(KERNEL, 2, __VA_ARGS__) }                                 \
    else { NU_J_CASES(KERNEL, 3, __VA_ARGS__) }

// a3: y = V grid
static int run_interp(nufft_plan_t p, int batch, const float2* grid, float2* y, cudaStream_t st) {
    if (p->M == 0) return NUFFT_OK;
    ProfScope ps(p, "interp", st);
    if (p->generic_j) {
        const dim3 blocks((unsigned)((p->M + 127) / 128), (unsigned)batch);
        NU_DJ_CASES(interp_direct_kernel, sample_data(p), grid_geom(p), grid, y, p->polyg)
        CU_TRY(cudaGetLastError());
        p->launches++;
        return NUFFT_OK;
    }
    if (p->d == 3 && (p->opts.interp_mode == 0 || p->opts.interp_mode == 3) && p->tile[0] == k3T0 && p->tile[1] == k3T1 && p->tile[2] == k3T2 && p->n_items > 0) {
        // tile-staged V (default tile only): register windows over pencil-sorted samples (win3d.cuh); interp_mode = 3 keeps
        // the half-warp-per-sample kernel of round 1, interp_mode = 1 the direct gather
        const dim3 tb((unsigned)p->n_items, (unsigned)batch);
        if (p->win3d && p->opts.interp_mode == 0) {
            CUtensorMap tm;
            const int use_tm = tile_tensor_map(p, batch, grid, &tm) ? 1 : 0;
            if (p->d_w3rec)
                interp_win_3d_kernel<kW3InterpWarps, true><<<tb, kW3InterpWarps * 32, win3d_smem(kW3InterpWarps), st>>>(
                    sample_data(p), grid_geom(p), p->d_items, grid, y, p->poly, tm, use_tm, p->d_w3rec);
            else
                interp_win_3d_kernel<kW3InterpWarps, false><<<tb, kW3InterpWarps * 32, win3d_smem(kW3InterpWarps), st>>>(
                    sample_data(p), grid_geom(p), p->d_items, grid, y, p->poly, tm, use_tm, nullptr);
        }
        else
            interp_tiled_3d_kernel<<<tb, 256, kInterp3dSmem, st>>>(sample_data(p), grid_geom(p), p->d_items, grid, y, p->poly);
        CU_TRY(cudaGetLastError());
        p->launches++;
        return NUFFT_OK;
    }
    if (p->d == 2 && p->opts.interp_mode == 0 && p->n_items > 0 && p->K[1] >= p->tg.pitch) {
        // tile-staged V: one CTA per V^H work item (the same tile-sorted sample ranges)
        const dim3 tb((unsigned)p->n_items, (unsigned)batch);
        CUtensorMap tm;
        const int use_tm = tile_tensor_map(p, batch, grid, &tm) ? 1 : 0;
        launch_pdl(interp_tiled_2d_kernel, tb, dim3(128), (size_t)p->tg.tile_cells * 8 + 16, st, sample_data(p), grid_geom(p), p->tg,
                   (const WorkItem*)p->d_items, grid, y, p->poly, tm, use_tm);
        CU_TRY(cudaGetLastError());
        p->launches++;
        return NUFFT_OK;
    }
    const dim3 blocks((unsigned)((p->M + 127) / 128), (unsigned)batch);
    if (p->d == 1) interp_direct_kernel<1><<<blocks, 128, 0, st>>>(sample_data(p), grid_geom(p), grid, y, p->poly);
    else if (p->d == 2) interp_direct_kernel<2><<<blocks, 128, 0, st>>>(sample_data(p), grid_geom(p), grid, y, p->poly);
    else           interp_direct_kernel<3><<<blocks, 128, 0, st>>>(sample_data(p), grid_geom(p), grid, y, p->poly);
    CU_TRY(cudaGetLastError());
    p->launches++;
    return NUFFT_OK;
}

// a4: grid = V^H y
static constexpr int kGrid2dWarps = 8;
static size_t smem_grid2d(nufft_plan_t p) { return (size_t)kGrid2dWarps * (size_t)grid2d_warp_bytes(p->tg.tile_cells); }
static size_t smem_grid3d(nufft_plan_t p) { return (size_t)p->tg.tile_cells * 8 + (size_t)kStage3dBytes; }

static int run_gridding(nufft_plan_t p, int batch, const float2* y, float2* grid, cudaStream_t st) {
    const bool det = p->opts.adjoint_mode == 1;
    if (p->M == 0 || p->n_items == 0) {
        CU_TRY(cudaMemsetAsync(grid, 0, (size_t)batch * p->cells * sizeof(float2), st));
        return NUFFT_OK;
    }
    if (p->generic_j && p->d == 2 && p->opts.adjoint_mode == 0 && p->K[1] >= p->tg.pitch) {
        // any width, 2-D: warp-private shared tiles + one TMA reduce-add flush per work item (gridding_tiled_2d_j_kernel)
        { ProfScope pz(p, "grid_zero", st); CU_TRY(cudaMemsetAsync(grid, 0, (size_t)batch * p->cells * sizeof(float2), st)); }
        ProfScope ps(p, "gridding", st);
        const dim3 blocks((unsigned)((p->n_items + kGrid2dWarps - 1) / kGrid2dWarps), (unsigned)batch);
#define NU_TILED_J(JJ) case JJ: gridding_tiled_2d_j_kernel<JJ><<<blocks, kGrid2dWarps * 32, (size_t)kGrid2dWarps * Tile2dJ<JJ>::warp_bytes(p->tg.tile_cells), st>>>( \
            sample_data(p), grid_geom(p), p->tg, p->d_items, p->n_items, y, grid, p->polyg); break;
        switch (p->J) {
            NU_TILED_J(2) NU_TILED_J(3) NU_TILED_J(4) NU_TILED_J(5) NU_TILED_J(6) NU_TILED_J(7) NU_TILED_J(8)
            default: return NUFFT_EINVAL;
        }
#undef NU_TILED_J
        CU_TRY(cudaGetLastError());
        p->launches++;
        return NUFFT_OK;
    }
    if (p->generic_j) {
        { ProfScope pz(p, "grid_zero", st); CU_TRY(cudaMemsetAsync(grid, 0, (size_t)batch * p->cells * sizeof(float2), st)); }
        ProfScope ps(p, "gridding", st);
        const dim3 blocks((unsigned)((p->M + 127) / 128), (unsigned)batch);
        NU_DJ_CASES(gridding_atomic_kernel, sample_data(p), grid_geom(p), y, grid, p->polyg)
        CU_TRY(cudaGetLastError());
        p->launches++;
        return NUFFT_OK;
    }
    const int64_t slab_stride = (int64_t)p->n_items * p->tg.tile_cells;
    if (det && !p->d_slabs)
        NU_TRY(dev_alloc((void**)&p->d_slabs, (size_t)p->max_batch * slab_stride * sizeof(float2), &p->bytes_work));
    if (!det) {
        ProfScope ps(p, "grid_zero", st);
        const int64_t n4 = (int64_t)batch * p->cells / 2;      // cells is even: float4 = two cells
        launch_pdl(grid_zero_kernel, dim3((unsigned)std::min<int64_t>((n4 + 255) / 256, 148 * 16)), dim3(256), 0, st, (float4*)grid, n4);
        CU_TRY(cudaGetLastError());
        p->launches++;
    }
    ProfScope ps(p, "gridding", st);
    if (p->d == 1) {       // 1-D: one thread per sample, one vector atomic per stencil point (the grid was zeroed above)
        const dim3 blocks((unsigned)((p->M + 127) / 128), (unsigned)batch);
        gridding_atomic_kernel<1><<<blocks, 128, 0, st>>>(sample_data(p), grid_geom(p), y, grid, p->poly);
    } else if (p->d == 2) {
        const dim3 blocks((unsigned)((p->n_items + kGrid2dWarps - 1) / kGrid2dWarps), (unsigned)batch);
        const size_t sm = smem_grid2d(p);
        CUtensorMap tm;
        const int use_tm = (!det && tile_tensor_map(p, batch, grid, &tm)) ? 1 : 0;
        if (det) { std::memset(&tm, 0, sizeof(tm)); gridding_tiled_2d_kernel<true><<<blocks, kGrid2dWarps * 32, sm, st>>>(sample_data(p), grid_geom(p), p->tg, p->d_items, p->n_items, y, grid, p->d_slabs, slab_stride, p->poly, tm, 0); }
        else     launch_pdl(gridding_tiled_2d_kernel<false>, blocks, dim3(kGrid2dWarps * 32), sm, st, sample_data(p), grid_geom(p), p->tg,
                            (const WorkItem*)p->d_items, p->n_items, y, grid, (float2*)nullptr, (int64_t)0, p->poly, tm, use_tm);
    } else if (!det && p->win3d && p->opts.adjoint_mode == 0) {
        const dim3 blocks((unsigned)p->n_items, (unsigned)batch);
        CUtensorMap tm;
        const int use_tm = tile_tensor_map(p, batch, grid, &tm) ? 1 : 0;
        if (p->d_w3rec)
            gridding_win_3d_kernel<kW3GridWarps, true><<<blocks, kW3GridWarps * 32, win3d_smem(kW3GridWarps), st>>>(
                sample_data(p), grid_geom(p), p->d_items, y, grid, p->poly, tm, use_tm, p->d_w3rec);
        else
            gridding_win_3d_kernel<kW3GridWarps, false><<<blocks, kW3GridWarps * 32, win3d_smem(kW3GridWarps), st>>>(
                sample_data(p), grid_geom(p), p->d_items, y, grid, p->poly, tm, use_tm, nullptr);
    } else {
        const dim3 blocks((unsigned)p->n_items, (unsigned)batch);
        const size_t sm = smem_grid3d(p);
        if (det) gridding_tiled_3d_kernel<true><<<blocks, 192, sm, st>>>(sample_data(p), grid_geom(p), p->tg, p->d_items, p->n_items, y, grid, p->d_slabs, slab_stride, p->poly);
        else     gridding_tiled_3d_kernel<false><<<blocks, 192, sm, st>>>(sample_data(p), grid_geom(p), p->tg, p->d_items, p->n_items, y, grid, nullptr, 0, p->poly);
    }
    CU_TRY(cudaGetLastError());
    p->launches++;
    if (det) {
        ProfScope pm(p, "gridding_merge", st);
        const dim3 blocks((unsigned)((p->cells + 255) / 256), (unsigned)batch);
        if (p->d == 2) gridding_merge_kernel<2><<<blocks, 256, 0, st>>>(grid_geom(p), p->tg, p->ntile[0], p->ntile[1], p->ntile[2], p->d_tile_item_start, p->d_slabs, slab_stride, grid);
        else           gridding_merge_kernel<3><<<blocks, 256, 0, st>>>(grid_geom(p), p->tg, p->ntile[0], p->ntile[1], p->ntile[2], p->d_tile_item_start, p->d_slabs, slab_stride, grid);
        CU_TRY(cudaGetLastError());
        p->launches++;
    }
    return NUFFT_OK;
}


// ------------------------------------------------------------------------------------------------------------
// batch-interleaved 2-D path (batch_il.cuh)
// ------------------------------------------------------------------------------------------------------------
static constexpr int kIlMinBatch = 12;    // measured crossover of the planar and interleaved paths
static bool use_il(nufft_plan_t p, int batch) { return p->il_ok && batch >= p->il_min_batch; }
static int il_groups(int batch) { return (batch + kIL - 1) / kIL; }

template <int K> static void launch_il_rows(bool adj, const IlRowParams& p, int blocks, cudaStream_t st) {
    constexpr int threads = FftGeom<K>::TPL * Rad<K>::TS;
    if (adj) launch_pdl(fft_il_rows_adj_kernel<K>, dim3(blocks), dim3(threads), smem_cols<K>(), st, p);
    else     launch_pdl(fft_il_rows_fwd_kernel<K>, dim3(blocks), dim3(threads), smem_cols<K>(), st, p);
}
static int dispatch_il_rows(int K, bool adj, const IlRowParams& p, cudaStream_t st) {
    const int T = tile_T(K);
    if (T == 0) return NUFFT_EINVAL;
    const int blocks = ((il_groups(p.batch) * kIL) / T) * p.n_outer;
    switch (K) {
        case 32: launch_il_rows<32>(adj, p, blocks, st); break;
        case 64: launch_il_rows<64>(adj, p, blocks, st); break;
        case 128: launch_il_rows<128>(adj, p, blocks, st); break;
        case 256: launch_il_rows<256>(adj, p, blocks, st); break;
        case 512: launch_il_rows<512>(adj, p, blocks, st); break;
        case 1024: launch_il_rows<1024>(adj, p, blocks, st); break;
        default: return NUFFT_EINVAL;
    }
    CU_TRY(cudaGetLastError());
    return NUFFT_OK;
}
template <int K> static void launch_il_rows_coilsum(const IlRowParams& p, cudaStream_t st) {
    constexpr int threads = FftGeom<K>::TPL * Rad<K>::TS;
    launch_pdl(fft_il_rows_adj_coilsum_kernel<K>, dim3(p.n_outer), dim3(threads), smem_cols<K>(), st, p);
}
static int dispatch_il_rows_coilsum(int K, const IlRowParams& p, cudaStream_t st) {
    switch (K) {
        case 32: launch_il_rows_coilsum<32>(p, st); break;
        case 64: launch_il_rows_coilsum<64>(p, st); break;
        case 128: launch_il_rows_coilsum<128>(p, st); break;
        case 256: launch_il_rows_coilsum<256>(p, st); break;
        case 512: launch_il_rows_coilsum<512>(p, st); break;
        case 1024: launch_il_rows_coilsum<1024>(p, st); break;
        default: return NUFFT_EINVAL;
    }
    CU_TRY(cudaGetLastError());
    return NUFFT_OK;
}
static IlRowParams il_row_params(nufft_plan_t p, int batch, const float2* img_in, float2* img_out, float2* grid,
                                 const float2* coil, bool same_image) {
    IlRowParams r{};
    r.img_in = img_in; r.img_out = img_out; r.grid = grid; r.coil = coil;
    r.s_outer = p->unit_scale ? p->d_ones : p->d_scale[0]; r.s_line = p->unit_scale ? p->d_ones : p->d_scale[1];
    r.tw = p->d_tw[1];
    r.n_outer = p->N[0]; r.k_outer = p->K[0]; r.batch = batch; r.same_image = same_image ? 1 : 0;
    return r;
}
static ColPassParams il_col_params(nufft_plan_t p, int batch, float2* grid) {
    ColPassParams c{};
    c.grid = grid; c.tw = p->d_tw[0];
    c.batch_stride = p->cells * kIL; c.outer_stride = 0; c.line_stride = (int64_t)p->K[1] * kIL;
    c.n_outer = 1; c.k_outer = 0; c.inner = p->K[1] * kIL;
    c.ngroups = il_groups(batch) * (c.inner / tile_T(p->K[0]));
    return c;
}
static IlPlan il_plan(nufft_plan_t p) {
    IlPlan s{};
    s.kpack = p->d_il_kpack; s.delta = p->d_il_delta; s.pos = p->d_il_pos; s.wtab = p->d_il_wtab;
    s.rowptr = p->d_il_rowptr; s.v2h = p->d_il_v2h;
    s.kpack_c = p->d_il_kpack_c; s.delta_c = p->d_il_delta_c;
    s.gbase = p->d_il_gbase; s.gbase_c = p->d_il_gbase_c;
    s.wv = p->d_il_wv; s.wv_c = p->d_il_wv_c;
    s.kpack_t = p->d_il_kpack_t; s.delta_t = p->d_il_delta_t; s.gbase_t = p->d_il_gbase_t; s.wv_t = p->d_il_wv_t; s.t2h = p->d_il_t2h;
    return s;
}

// a1 + a2 on the interleaved grid
static int run_scale_fft_il(nufft_plan_t p, int batch, const float2* x, float2* grid, const float2* coil,
                            bool same_image, cudaStream_t st) {
    IlRowParams r = il_row_params(p, batch, x, nullptr, grid, coil, same_image);
    { ProfScope ps(p, "fft_rows_fwd", st); NU_TRY(dispatch_il_rows(p->K[1], false, r, st)); }
    { ProfScope ps(p, "fft_cols_fwd", st); NU_TRY(dispatch_cols(p->K[0], false, il_col_params(p, batch, grid), st)); }
    p->launches += 2;
    return NUFFT_OK;
}
// a5 + a6 on the interleaved grid
static int run_fft_scale_il(nufft_plan_t p, int batch, float2* grid, float2* x, const float2* coil, cudaStream_t st,
                            bool coil_sum = false) {
    PdlOff no_pdl;
    {
        ColPassParams c = il_col_params(p, batch, grid);
        c.mult = p->cur_mult; c.mult_shift = 5;
        ProfScope ps(p, "fft_cols_adj", st);
        NU_TRY(dispatch_cols(p->K[0], true, c, st));
    }
    IlRowParams r = il_row_params(p, batch, nullptr, x, grid, coil, false);
    if (coil_sum) {      // x is the coil-summed image [N0][N1] (eq. 35): the sum is fused into the last pass
        ProfScope ps(p, "fft_rows_adj", st);
        NU_TRY(dispatch_il_rows_coilsum(p->K[1], r, st));
    } else {
        ProfScope ps(p, "fft_rows_adj", st);
        NU_TRY(dispatch_il_rows(p->K[1], true, r, st));
    }
    p->launches += 2;
    return NUFFT_OK;
}
// a3: y_il[group][sorted sample][32] = V grid_il
static int run_interp_il(nufft_plan_t p, int batch, const float2* grid, float2* y_il, cudaStream_t st) {
    if (p->M == 0) return NUFFT_OK;
    const dim3 blocks((unsigned)((p->M + kInterpChunk - 1) / kInterpChunk), (unsigned)il_groups(batch));
    ProfScope ps(p, "interp", st);
    if (p->n_il_titems > 0) {     // register windows fed from shared tiles (interp_mode = 0)
        using G = IlTile<kItT, kItWarps>;
        const int ng = il_groups(batch);
        CUtensorMap tm;
        std::memset(&tm, 0, sizeof(tm));
        int use_tm = 0;
        if (tmap_encode_fn enc = tmap_encoder()) {      // grid_il [groups][K0][K1][32] complex64 as float32 [groups][K0][K1][64]
            const cuuint32_t est[4] = {1, 1, 1, 1};
            const cuuint64_t gdim[4] = {(cuuint64_t)2 * kIL, (cuuint64_t)p->K[1], (cuuint64_t)p->K[0], (cuuint64_t)ng};
            const cuuint64_t gstr[3] = {(cuuint64_t)kIL * 8, (cuuint64_t)p->K[1] * kIL * 8, (cuuint64_t)p->cells * kIL * 8};
            const cuuint32_t box[4] = {2 * kIL, (cuuint32_t)G::PW, (cuuint32_t)G::PW, 1};
            use_tm = enc(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (void*)grid, gdim, gstr, box, est, CU_TENSOR_MAP_INTERLEAVE_NONE,
                         CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS ? 1 : 0;
        }
        launch_pdl(interp_il_tile_kernel<kItT, kItWarps, 2>, dim3((unsigned)(p->n_il_titems * ng)), dim3(kItWarps * 32), (size_t)G::SMEM, st,
                   il_plan(p), grid_geom(p), (const IlTileItem*)p->d_il_titems, p->n_il_titems, ng, grid, y_il, p->poly, tm, use_tm);
    } else
    if (p->opts.interp_mode != 3) {     // register windows over the block-sorted walk (interp_mode = 3: round-1 kernel)
        const dim3 wb((unsigned)((p->M + kIwWarps * 32 - 1) / (kIwWarps * 32)), (unsigned)il_groups(batch));
        launch_pdl(interp_il_win_kernel<false>, wb, dim3(kIwWarps * 32), 0, st, il_plan(p), grid_geom(p), grid, y_il, batch, p->poly);
    } else
    interp_il_kernel<false, kInterpChunk><<<blocks, 256, 0, st>>>(il_plan(p), grid_geom(p), grid, y_il, batch, p->poly);
    CU_TRY(cudaGetLastError());
    p->launches++;
    return NUFFT_OK;
}
// a3 for trajectory-coherent plans: y[batch][M] in the caller's order straight from the kernel (no layout pass)
static int run_interp_il_caller(nufft_plan_t p, int batch, const float2* grid, float2* y, cudaStream_t st) {
    if (p->M == 0) return NUFFT_OK;
    const dim3 blocks((unsigned)((p->M + kInterpChunkCaller - 1) / kInterpChunkCaller), (unsigned)il_groups(batch));
    ProfScope ps(p, "interp", st);
    if (p->opts.interp_mode != 3) {
        const dim3 wb((unsigned)((p->M + kIwWarps * 32 - 1) / (kIwWarps * 32)), (unsigned)il_groups(batch));
        launch_pdl(interp_il_win_kernel<true>, wb, dim3(kIwWarps * 32), 0, st, il_plan(p), grid_geom(p), grid, y, batch, p->poly);
    } else
    interp_il_kernel<true, kInterpChunkCaller><<<blocks, 256, 0, st>>>(il_plan(p), grid_geom(p), grid, y, batch, p->poly);
    CU_TRY(cudaGetLastError());
    p->launches++;
    return NUFFT_OK;
}
// caller's y[batch][M] -> d_yil
static int run_y_to_il(nufft_plan_t p, int batch, const float2* y, cudaStream_t st) {
    PdlOff no_pdl;
    if (p->M == 0) return NUFFT_OK;
    if (!p->d_yil)
        NU_TRY(dev_alloc((void**)&p->d_yil, (size_t)p->batch_pad * p->M * sizeof(float2), &p->bytes_work));
    const dim3 blocks((unsigned)((p->M + 127) / 128), (unsigned)il_groups(batch));
    ProfScope ps(p, "y_to_il", st);
    launch_pdl(y_to_il_kernel, blocks, dim3(128), 0, st, (const int32_t*)p->d_il_pos, y, p->d_yil, p->M, batch);
    CU_TRY(cudaGetLastError());
    p->launches++;
    return NUFFT_OK;
}
// y_il -> caller's y[batch][M]
static int run_y_from_il(nufft_plan_t p, int batch, const float2* y_il, float2* y, cudaStream_t st) {
    if (p->M == 0) return NUFFT_OK;
    const dim3 blocks((unsigned)((p->M + 127) / 128), (unsigned)il_groups(batch));
    ProfScope ps(p, "y_from_il", st);
    launch_pdl(y_from_il_kernel, blocks, dim3(128), 0, st, (const int32_t*)p->d_il_pos, y_il, y, p->M, batch);
    CU_TRY(cudaGetLastError());
    p->launches++;
    return NUFFT_OK;
}
// a4 from y_il
static int run_gridding_il(nufft_plan_t p, int batch, const float2* y_il, float2* grid, cudaStream_t st) {
    PdlOff no_pdl;
    if (p->M == 0) {
        CU_TRY(cudaMemsetAsync(grid, 0, (size_t)il_groups(batch) * kIL * p->cells * sizeof(float2), st));
        return NUFFT_OK;
    }
    const int ng = il_groups(batch);
    ProfScope ps(p, "gridding", st);
    // CTAs handle two groups (64 images) at a time: the staged weight records and row lookups are shared
    if (ng >= 2) {
        const dim3 blocks((unsigned)p->n_il_items, (unsigned)(ng / 2));
        launch_pdl(gridding_il_kernel<2>, blocks, dim3(256), GridStage<2>::BYTES, st, il_plan(p), grid_geom(p), (const IlItem*)p->d_il_items, y_il, grid, 0);
        p->launches++;
    }
    if (ng & 1) {
        const dim3 blocks((unsigned)p->n_il_items, 1u);
        launch_pdl(gridding_il_kernel<1>, blocks, dim3(256), GridStage<1>::BYTES, st, il_plan(p), grid_geom(p), (const IlItem*)p->d_il_items, y_il, grid, ng - 1);
        p->launches++;
    }
    CU_TRY(cudaGetLastError());
    return NUFFT_OK;
}

// ------------------------------------------------------------------------------------------------------------
// plan
// ------------------------------------------------------------------------------------------------------------
static bool supported_K(int64_t K) { return K == 32 || K == 64 || K == 128 || K == 256 || K == 512 || K == 1024; }

template <class T> static int dev_upload(T** dptr, const std::vector<T>& h, int64_t* bytes) {
    *dptr = nullptr;
    if (h.empty()) return NUFFT_OK;
    cudaError_t e = cudaMalloc((void**)dptr, h.size() * sizeof(T));
    if (e != cudaSuccess) { g_last_cuda_error = (int)e; (void)cudaGetLastError(); return e == cudaErrorMemoryAllocation ? NUFFT_ENOMEM : NUFFT_ECUDA; }
    CU_TRY(cudaMemcpy(*dptr, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice));
    if (bytes) *bytes += (int64_t)(h.size() * sizeof(T));
    return NUFFT_OK;
}
static int dev_alloc(void** dptr, size_t bytes, int64_t* acct) {
    *dptr = nullptr;
    if (bytes == 0) return NUFFT_OK;
    cudaError_t e = cudaMalloc(dptr, bytes);
    if (e != cudaSuccess) { g_last_cuda_error = (int)e; (void)cudaGetLastError(); return e == cudaErrorMemoryAllocation ? NUFFT_ENOMEM : NUFFT_ECUDA; }
    if (acct) *acct += (int64_t)bytes;
    return NUFFT_OK;
}

extern "C" int nufft_default_opts(nufft_opts* o) {
    if (!o) return NUFFT_EINVAL;
    std::memset(o, 0, sizeof(*o));
    return NUFFT_OK;
}

// Plan data of the batch-interleaved path (batch_il.cuh).  Two sample orders:
//   V order   key (column band, row k0_0, column)          consecutive samples share stencil rows: L1 reuse in interp_il
//   V^H order key (column band, class, row k0_0, column)   class 0 = column offset in the band >= 3 (stencil reaches into
//             the next band), class 1 = the rest.  For one output row of one band the contributing samples are then
//             three contiguous ranges (this band class 0, this band class 1, previous band class 0), each sorted by row.
// y_il (the interleaved sample vectors) always uses the V^H order.
static int plan_build_il(nufft_plan_t p, const std::vector<uint32_t>& kpack, const std::vector<float>& delta,
                         const std::vector<double>& delta64) {
    const int64_t M = p->M;
    const int K0 = p->K[0], K1 = p->K[1], nb = K1 / kBandW;
    const double J = (double)kJ, beta = host::kb_beta(J, 2.0);
    auto row_of = [](uint32_t kp) { return (int)(kp & 1023u); };
    auto col_of = [](uint32_t kp) { return (int)((kp >> 10) & 1023u); };
    // counting sort by a key function over nbins bins; returns perm (sorted position -> caller sample) and bin starts
    auto sort_by = [&](auto key_of, int64_t nbins, std::vector<int32_t>& perm, std::vector<int32_t>& binstart) {
        binstart.assign(nbins + 1, 0);
        for (int64_t m = 0; m < M; ++m) binstart[key_of(kpack[m]) + 1]++;
        for (int64_t b = 0; b < nbins; ++b) binstart[b + 1] += binstart[b];
        perm.resize(M);
        std::vector<int32_t> cur(binstart.begin(), binstart.end() - 1);
        for (int64_t m = 0; m < M; ++m) perm[cur[key_of(kpack[m])]++] = (int32_t)m;
    };
    // ---- V order
    std::vector<int32_t> perm_v, bins_v;
    const int nbr = (K0 + 2) / 3, nbc = (K1 + 2) / 3;     // 3 x 3 blocks of stencil base cells, column-block major
    sort_by([&](uint32_t kp) -> int64_t {
        const int r = row_of(kp), c = col_of(kp);
        return ((int64_t)(c / 3) * nbr + r / 3) * 9 + (r % 3) * 3 + (c % 3);
    }, (int64_t)nbc * nbr * 9, perm_v, bins_v);
    // window groups of a walk order (interp_il_win_kernel): the order is cut into runs of consecutive samples whose stencil
    // bases fit the span of a window shape (rows x columns of cells: 8x8, 6x10, 10x6, 7x9, 9x7 -> base spans 2x2, 0x4, 4x0,
    // 1x3, 3x1); greedily, the shape with the fewest window cells per sample wins.  Runs never cross a 32-sample boundary
    // (one warp walks 32 consecutive samples) and never wrap.  Every sample records base row | base column << 10 | shape << 20.
    auto window_groups = [&](auto kp_at, std::vector<uint32_t>& gb) {
        gb.resize(M);
        int64_t i = 0;
        while (i < M) {
            const int64_t cap = 32 - (i % 32);
            int best_sh = 0, best_lo0 = 0, best_lo1 = 0;
            int64_t best_n = 0;
            for (int sh = 0; sh < kIwShapes; ++sh) {
                const int sp0 = iw_rows(sh) - kJ, sp1 = iw_cols(sh) - kJ;
                int lo0 = row_of(kp_at(i)), hi0 = lo0, lo1 = col_of(kp_at(i)), hi1 = lo1;
                int64_t j = i + 1;
                for (; j < M && j - i < cap; ++j) {
                    const int r = row_of(kp_at(j)), c = col_of(kp_at(j));
                    const int nlo0 = std::min(lo0, r), nhi0 = std::max(hi0, r), nlo1 = std::min(lo1, c), nhi1 = std::max(hi1, c);
                    if (nhi0 - nlo0 > sp0 || nhi1 - nlo1 > sp1) break;
                    lo0 = nlo0; hi0 = nhi0; lo1 = nlo1; hi1 = nhi1;
                }
                const int64_t n = j - i;
                // cells per sample: rows * cols / n, compared by cross-multiplication (all shapes hold 60-64 cells)
                if (best_n == 0 || (int64_t)iw_rows(sh) * iw_cols(sh) * best_n < (int64_t)iw_rows(best_sh) * iw_cols(best_sh) * n) {
                    best_n = n; best_sh = sh; best_lo0 = lo0; best_lo1 = lo1;
                }
            }
            const uint32_t base = (uint32_t)best_lo0 | ((uint32_t)best_lo1 << 10) | ((uint32_t)best_sh << 20);
            for (int64_t k = i; k < i + best_n; ++k) gb[k] = base;
            i += best_n;
        }
    };
    // ---- V^H order: bins (band, class, row)
    std::vector<int32_t> perm_h, rowptr;
    sort_by([&](uint32_t kp) -> int64_t {
        const int r = row_of(kp), c = col_of(kp);
        return ((int64_t)(c / kBandW) * 2 + ((c % kBandW) >= 3 ? 0 : 1)) * K0 + r;
    }, (int64_t)nb * 2 * K0, perm_h, rowptr);
    // rowptr[(band*2 + class) * K0 + r] .. [.. + r + 1]: samples of (band, class, row r); classes are adjacent, so the entry
    // one past the last row of a class is the start of the next class / band.
    std::vector<int32_t> pos_h(M);
    for (int64_t i = 0; i < M; ++i) pos_h[perm_h[i]] = (int32_t)i;
    std::vector<uint32_t> kp_s(M);
    std::vector<float> dl_s((size_t)2 * M);
    std::vector<int32_t> v2h(M);
    for (int64_t i = 0; i < M; ++i) {
        const int64_t m = perm_v[i];
        kp_s[i] = kpack[m];
        dl_s[i] = delta[m];
        dl_s[M + i] = delta[M + m];
        v2h[i] = pos_h[m];
    }
    // coef_mode = 1: the zero-padded weight vectors of interp_il_win_kernel, float64-built, per walk order
    auto weight_table = [&](auto sample_at, const std::vector<uint32_t>& gb, std::vector<float>& tab) {
        tab.assign((size_t)M * 24, 0.f);
        for (int64_t i = 0; i < M; ++i) {
            const int64_t m = sample_at(i);
            double w0[kJ], w1[kJ];
            if (p->minmax) { p->mm[0].weights(delta64[m], w0); p->mm[1].weights(delta64[M + m], w1); }
            else { host::kb_weights_f64(delta64[m], J, beta, w0); host::kb_weights_f64(delta64[M + m], J, beta, w1); }
            const int o0 = row_of(kpack[m]) - (int)(gb[i] & 1023u), o1 = col_of(kpack[m]) - (int)((gb[i] >> 10) & 1023u);
            for (int j = 0; j < kJ; ++j) { tab[(size_t)i * 24 + o0 + j] = (float)w0[j]; tab[(size_t)i * 24 + 12 + o1 + j] = (float)w1[j]; }
        }
    };
    std::vector<float> wtab((size_t)M * kTabW, 0.f);
    for (int64_t i = 0; i < M; ++i) {
        const int64_t m = perm_h[i];
        double w0[kJ], w1[kJ];
        if (p->minmax) { p->mm[0].weights(delta64[m], w0); p->mm[1].weights(delta64[M + m], w1); }
        else { host::kb_weights_f64(delta64[m], J, beta, w0); host::kb_weights_f64(delta64[M + m], J, beta, w1); }
        float* rec = &wtab[(size_t)i * kTabW];
        const int32_t r = row_of(kpack[m]);
        for (int j = 0; j < kJ; ++j) rec[(r + j) & 7] = (float)w0[j];     // rotated by the base row: output row R reads slot R & 7
        const int off = col_of(kpack[m]) % kBandW;
        for (int j = 0; j < kJ; ++j) {
            const int c = off + j;                       // column relative to the start of the sample's own band
            if (c < kBandW) rec[8 + c] = (float)w1[j];   // part A: this band
            else rec[16 + c - kBandW] = (float)w1[j];    // part B: the next band
        }
    }
    // work items: blocks of 8 rows; rows whose interaction count is far above the mean are split among warps
    auto cnt_rows = [&](int cb, int cls, int r_lo, int r_hi) -> int64_t {      // rows r_lo..r_hi inclusive, no wrap
        const size_t base = ((size_t)cb * 2 + cls) * K0;
        return rowptr[base + r_hi + 1] - rowptr[base + r_lo];
    };
    std::vector<int64_t> rowload((size_t)nb * K0);
    int64_t total = 0;
    for (int cb = 0; cb < nb; ++cb) {
        const int cbp = (cb + nb - 1) % nb;
        for (int r = 0; r < K0; ++r) {
            int64_t l = 0;
            auto add = [&](int lo, int hi) { l += cnt_rows(cb, 0, lo, hi) + cnt_rows(cb, 1, lo, hi) + cnt_rows(cbp, 0, lo, hi); };
            if (r >= kJ - 1) add(r - (kJ - 1), r);
            else { add(0, r); add(K0 - (kJ - 1) + r, K0 - 1); }
            rowload[(size_t)cb * K0 + r] = l;
            total += l;
        }
    }
    const int64_t thr = std::max<int64_t>(192, 3 * total / std::max<int64_t>(1, (int64_t)nb * K0));
    std::vector<IlItem> items;
    for (int cb = 0; cb < nb; ++cb)
        for (int r0 = 0; r0 < K0; r0 += 8) {
            int64_t mx = 0;
            for (int r = r0; r < r0 + 8; ++r) mx = std::max(mx, rowload[(size_t)cb * K0 + r]);
            int nrows = 8;
            while (nrows > 1 && mx * nrows / 8 > thr) nrows /= 2;     // per-warp share of the heaviest row
            for (int q = 0; q < 8; q += nrows) {
                int64_t l = 0;
                for (int r = r0 + q; r < r0 + q + nrows; ++r) l += rowload[(size_t)cb * K0 + r];
                items.push_back(IlItem{cb, r0 + q, nrows, (int32_t)std::min<int64_t>(l, 0x7fffffff)});
            }
        }
    std::stable_sort(items.begin(), items.end(), [](const IlItem& a, const IlItem& b) { return a.load > b.load; });
    p->n_il_items = (int)items.size();
    // trajectory coherence of the caller's order: consecutive samples within two cells of each other on both axes
    // (modulo the grid) in at least 90 % of the cases -> V can walk the caller's order and write y directly
    {
        int64_t near = 0;
        for (int64_t m = 1; m < M; ++m) {
            int d0 = std::abs(row_of(kpack[m]) - row_of(kpack[m - 1])), d1 = std::abs(col_of(kpack[m]) - col_of(kpack[m - 1]));
            d0 = std::min(d0, K0 - d0); d1 = std::min(d1, K1 - d1);
            near += (d0 <= 2 && d1 <= 2) ? 1 : 0;
        }
        p->il_coherent = (M > 1) && (near * 10 >= (M - 1) * 9) && (p->opts.interp_mode == 0 || p->opts.interp_mode == 3);
        if (p->il_coherent) {
            std::vector<uint32_t> gb_c;
            window_groups([&](int64_t i) { return kpack[i]; }, gb_c);
            NU_TRY(dev_upload(&p->d_il_kpack_c, kpack, &p->bytes_plan));
            NU_TRY(dev_upload(&p->d_il_delta_c, delta, &p->bytes_plan));
            NU_TRY(dev_upload(&p->d_il_gbase_c, gb_c, &p->bytes_plan));
            if (p->opts.coef_mode == 1) {
                std::vector<float> tab;
                weight_table([&](int64_t i) { return i; }, gb_c, tab);
                NU_TRY(dev_upload(&p->d_il_wv_c, tab, &p->bytes_plan));
            }
        }
    }
    {
        std::vector<uint32_t> gb_v;
        window_groups([&](int64_t i) { return kp_s[i]; }, gb_v);
        NU_TRY(dev_upload(&p->d_il_gbase, gb_v, &p->bytes_plan));
        if (p->opts.coef_mode == 1) {
            std::vector<float> tab;
            weight_table([&](int64_t i) { return (int64_t)perm_v[i]; }, gb_v, tab);
            NU_TRY(dev_upload(&p->d_il_wv, tab, &p->bytes_plan));
        }
    }
    // ---- tile order (interp_il_tile_kernel): samples sorted by tile of kItT x kItT base cells, inside a tile by 3 x 3 blocks
    // relative to the tile origin; work items of <= kItWarps * 32 samples (a tile with more is cut into equal parts); warp w of
    // an item walks its w-th share, and window groups never cross a share.  Window bases are stored relative to the tile
    // origin and clamped so that the window stays inside the padded tile.
    if (p->opts.interp_mode == 0 && K0 >= IlTile<kItT, kItWarps>::PW && K1 >= IlTile<kItT, kItWarps>::PW) {
        constexpr int T = kItT, PW = IlTile<kItT, kItWarps>::PW, CAP = IlTile<kItT, kItWarps>::CAP, NB = (T + 2) / 3;
        const int ntr = (K0 + T - 1) / T, ntc = (K1 + T - 1) / T;
        const int64_t per_tile = (int64_t)NB * NB * 9;
        std::vector<int32_t> perm_t, bins_t;
        sort_by([&](uint32_t kp) -> int64_t {
            const int r = row_of(kp), c = col_of(kp), rr = r % T, cc = c % T;
            return ((int64_t)(c / T) * ntr + r / T) * per_tile + ((int64_t)(cc / 3) * NB + rr / 3) * 9 + (rr % 3) * 3 + (cc % 3);
        }, (int64_t)ntr * ntc * per_tile, perm_t, bins_t);
        std::vector<uint32_t> kp_t(M), gb_t(M);
        std::vector<float> dl_t((size_t)2 * M);
        std::vector<int32_t> t2h(M);
        for (int64_t i = 0; i < M; ++i) {
            const int64_t m = perm_t[i];
            kp_t[i] = kpack[m]; dl_t[i] = delta[m]; dl_t[M + i] = delta[M + m]; t2h[i] = pos_h[m];
        }
        std::vector<IlTileItem> titems;
        for (int tc = 0; tc < ntc; ++tc)
            for (int tr = 0; tr < ntr; ++tr) {
                const int64_t tb = ((int64_t)tc * ntr + tr) * per_tile;
                const int64_t a = bins_t[tb], n = bins_t[tb + per_tile] - a;
                if (n == 0) continue;
                const int64_t parts = (n + CAP - 1) / CAP;
                for (int64_t q = 0; q < parts; ++q) {
                    const int64_t lo = a + n * q / parts, hi = a + n * (q + 1) / parts;
                    titems.push_back(IlTileItem{(int32_t)lo, (int32_t)(hi - lo), tr * T, tc * T});
                }
            }
        for (const IlTileItem& it : titems) {
            const int per = (it.cnt + kItWarps - 1) / kItWarps;
            for (int w = 0; w < kItWarps; ++w) {
                const int64_t lo = it.start + (int64_t)w * per, hi = std::min<int64_t>((int64_t)it.start + it.cnt, lo + per);
                int64_t i = lo;
                while (i < hi) {      // greedy runs whose bases fit a 3 x 3 box: one 8 x 8 window (measured: the other shapes of
                    // interp_il_win gain nothing in this order)
                    int lo0 = row_of(kp_t[i]), hi0 = lo0, lo1 = col_of(kp_t[i]), hi1 = lo1;
                    int64_t j = i + 1;
                    for (; j < hi; ++j) {
                        const int r = row_of(kp_t[j]), c = col_of(kp_t[j]);
                        const int nlo0 = std::min(lo0, r), nhi0 = std::max(hi0, r), nlo1 = std::min(lo1, c), nhi1 = std::max(hi1, c);
                        if (nhi0 - nlo0 > kItWin - kJ || nhi1 - nlo1 > kItWin - kJ) break;
                        lo0 = nlo0; hi0 = nhi0; lo1 = nlo1; hi1 = nhi1;
                    }
                    const int b0 = std::min(lo0 - it.r0, PW - kItWin), b1 = std::min(lo1 - it.c0, PW - kItWin);
                    const uint32_t base = (uint32_t)b0 | ((uint32_t)b1 << 5);
                    for (int64_t k = i; k < j; ++k) gb_t[k] = base;
                    i = j;
                }
            }
        }
        std::stable_sort(titems.begin(), titems.end(), [](const IlTileItem& a, const IlTileItem& b) { return a.cnt > b.cnt; });
        p->n_il_titems = (int)titems.size();
        NU_TRY(dev_upload(&p->d_il_kpack_t, kp_t, &p->bytes_plan));
        NU_TRY(dev_upload(&p->d_il_delta_t, dl_t, &p->bytes_plan));
        NU_TRY(dev_upload(&p->d_il_gbase_t, gb_t, &p->bytes_plan));
        NU_TRY(dev_upload(&p->d_il_t2h, t2h, &p->bytes_plan));
        NU_TRY(dev_upload(&p->d_il_titems, titems, &p->bytes_plan));
        if (p->opts.coef_mode == 1) {
            std::vector<float> tab((size_t)M * 12, 0.f);
            for (int64_t i = 0; i < M; ++i) {
                const int64_t m = perm_t[i];
                double w0[kJ], w1[kJ];
                if (p->minmax) { p->mm[0].weights(delta64[m], w0); p->mm[1].weights(delta64[M + m], w1); }
                else { host::kb_weights_f64(delta64[m], J, beta, w0); host::kb_weights_f64(delta64[M + m], J, beta, w1); }
                for (int j = 0; j < kJ; ++j) { tab[(size_t)i * 12 + j] = (float)w0[j]; tab[(size_t)i * 12 + 6 + j] = (float)w1[j]; }
            }
            NU_TRY(dev_upload(&p->d_il_wv_t, tab, &p->bytes_plan));
        }
    }
    NU_TRY(dev_upload(&p->d_il_kpack, kp_s, &p->bytes_plan));
    NU_TRY(dev_upload(&p->d_il_delta, dl_s, &p->bytes_plan));
    NU_TRY(dev_upload(&p->d_il_v2h, v2h, &p->bytes_plan));
    NU_TRY(dev_upload(&p->d_il_pos, pos_h, &p->bytes_plan));
    NU_TRY(dev_upload(&p->d_il_wtab, wtab, &p->bytes_plan));
    NU_TRY(dev_upload(&p->d_il_rowptr, rowptr, &p->bytes_plan));
    NU_TRY(dev_upload(&p->d_il_items, items, &p->bytes_plan));
    return NUFFT_OK;
}

static int plan_build(nufft_plan_t p, const double* om) {
    const int d = p->d;
    const double J = (double)p->J;
    // kernel polynomial, scaling vectors, twiddles (float64 on the host, rounded once)
    p->poly_err = 0.0;
    for (int a = 0; a < d; ++a) {       // one kernel shape per axis: sigma_a = K_a / N_a (and N_a itself for min-max)
        double err = 0.0;
        const double sigma = (double)p->K[a] / (double)p->N[a];
        if (p->minmax) {
            p->mm[a].build(p->N[a], p->K[a], p->J);
            if (p->generic_j) p->mm[a].fit_axis(p->polyg, a, &err);
            else p->mm[a].fit_axis(p->poly, a, &err);
        } else if (p->generic_j) host::fit_kernel_axis(p->polyg, a, p->J, sigma, &err);
        else host::fit_kernel_axis(p->poly, a, p->J, sigma, &err);
        p->poly_err = std::max(p->poly_err, err);
    }
    for (int a = 0; a < d; ++a) {
        NU_TRY(dev_upload(&p->d_scale[a], host::scaling_vector(p->N[a], p->K[a], J), &p->bytes_plan));
        NU_TRY(dev_upload(&p->d_tw[a], host::twiddle_table(p->K[a]), &p->bytes_plan));
    }
    {
        int nmax = 1;
        for (int a = 0; a < d; ++a) nmax = std::max(nmax, p->N[a]);
        NU_TRY(dev_upload(&p->d_ones, std::vector<float>((size_t)nmax, 1.0f), &p->bytes_plan));
    }
    // tiles
    const int def1[3] = {32, 1, 1}, def2[3] = {16, 32, 1}, def3[3] = {8, 8, 16};
    for (int a = 0; a < 3; ++a) {
        int t = (a < d) ? p->opts.tile[a] : 1;
        if (a < d && t <= 0) t = std::min((d == 1) ? def1[a] : ((d == 2) ? def2[a] : def3[a]), p->K[a]);
        if (a < d && (t < 8 || t > p->K[a] || (p->K[a] % t) != 0 || (t & 1))) return NUFFT_EINVAL;
        p->tile[a] = t;
        p->ntile[a] = (a < d) ? p->K[a] / t : 1;
    }
    p->n_tiles = (int64_t)p->ntile[0] * p->ntile[1] * p->ntile[2];
    {
        TileGeom& tg = p->tg;
        // halo of J - 1 cells: the plan's own width on 2-D generic-width plans (gridding_tiled_2d_j_kernel), kJ otherwise
        const int Jt = (p->generic_j && d == 2) ? p->J : kJ;
        for (int a = 0; a < 3; ++a) { tg.T[a] = p->tile[a]; tg.P[a] = (a < d) ? p->tile[a] + Jt - 1 : 1; }
        // row pitch: >= T + J (8-cell aligned windows reach one cell past the halo) and = 8 (mod 16) cells, so that the
        // two stencil rows of an 8-lane shared-memory phase fall into different 64-byte bank halves
        int pitch = p->tile[d - 1] + Jt;
        pitch += ((8 - pitch % 16) + 16) % 16;
        tg.pitch = pitch;
        tg.plane = (d == 3) ? tg.P[1] * pitch : 0;
        tg.tile_cells = (d == 3) ? tg.P[0] * tg.P[1] * pitch : tg.P[0] * pitch;
        // a user tile whose shared-memory footprint exceeds the opt-in (200 KB) would fail at every adjoint launch
        const size_t need = (d == 3) ? (size_t)tg.tile_cells * 8 + (size_t)kStage3dBytes
                                     : (d == 2 ? (size_t)8 * (size_t)grid2d_warp_bytes(tg.tile_cells) : 0);
        if (need > (size_t)200 * 1024) return NUFFT_EINVAL;
    }
    // per-sample split (float64) and tile id
    const int64_t M = p->M;
    std::vector<uint32_t> kpack(M);
    std::vector<float> delta((size_t)d * M);
    const bool want64 = p->il_ok || p->opts.coef_mode == 1;
    std::vector<double> delta64(want64 ? (size_t)d * M : 0);
    // 3-D, J = 6, default tile: inside a tile the samples are sorted by pencil (3 x 3 block of stencil base cells on axes
    // 0, 1) and base pair on axis 2, the order the register-window kernels of win3d.cuh walk
    p->win3d = (d == 3) && !p->generic_j && p->tile[0] == k3T0 && p->tile[1] == k3T1 && p->tile[2] == k3T2;
    const int nsub = p->win3d ? kW3SubKeys : 1;
    std::vector<int64_t> tid(M);        // tile id * nsub + key inside the tile
    for (int64_t m = 0; m < M; ++m) {
        uint32_t kp = 0;
        int64_t t = 0;
        int c[3] = {0, 0, 0};
        for (int a = 0; a < d; ++a) {
            const double w = om[m * d + a];
            if (!std::isfinite(w)) return NUFFT_ERANGE;
            float df;
            double d64;
            const int k0 = host::split_coordinate(w, p->K[a], J, &df, &d64);
            if (want64) delta64[(size_t)a * M + m] = d64;
            kp |= (uint32_t)k0 << (10 * a);
            delta[(size_t)a * M + m] = df;
            t = t * p->ntile[a] + k0 / p->tile[a];
            c[a] = k0 % p->tile[a];
        }
        kpack[m] = kp;
        tid[m] = t * nsub + (p->win3d ? w3_sub_key(c[0], c[1], c[2]) : 0);
    }
    // stable counting sort by (tile, key inside the tile)
    std::vector<int64_t> start(p->n_tiles + 1, 0);
    std::vector<int32_t> perm(M);
    {
        std::vector<int64_t> fine((size_t)p->n_tiles * nsub + 1, 0);
        for (int64_t m = 0; m < M; ++m) fine[tid[m] + 1]++;
        for (size_t b = 0; b + 1 < fine.size(); ++b) fine[b + 1] += fine[b];
        for (int64_t t = 0; t <= p->n_tiles; ++t) start[t] = fine[(size_t)t * nsub];
        p->max_tile_samples = 0;
        for (int64_t t = 0; t < p->n_tiles; ++t) {
            const int64_t n = start[t + 1] - start[t];
            p->max_tile_samples = std::max<int64_t>(p->max_tile_samples, n);
            int k = 0;
            while (k + 1 < NUFFT_TILE_HIST_BUCKETS && ((int64_t)1 << k) <= n) ++k;      // n = 0 -> 0; 2^(k-1) <= n < 2^k -> k
            p->tile_hist[k]++;
        }
        for (int64_t m = 0; m < M; ++m) perm[fine[tid[m]]++] = (int32_t)m;
    }
    std::vector<uint32_t> kpack_s(M);
    std::vector<float> delta_s((size_t)d * M);
    for (int64_t i = 0; i < M; ++i) {
        kpack_s[i] = kpack[perm[i]];
        for (int a = 0; a < d; ++a) delta_s[(size_t)a * M + i] = delta[(size_t)a * M + perm[i]];
    }
    NU_TRY(dev_upload(&p->d_kpack, kpack_s, &p->bytes_plan));
    NU_TRY(dev_upload(&p->d_delta, delta_s, &p->bytes_plan));
    NU_TRY(dev_upload(&p->d_perm, perm, &p->bytes_plan));
    // coef_mode = 1 (north star item 3 "precomputed in a coalesced per-sample layout"): the records the
    // register-window 3-D kernels otherwise build on the fly (win3d.cuh w3_stage), evaluated here in float64 and rounded once,
    // in walk order: 112 contiguous bytes per sample, moved into shared memory by one bulk copy per 16 samples
    if (p->opts.coef_mode == 1 && p->win3d && M > 0) {
        std::vector<float> recs((size_t)M * kW3Rec, 0.f);
        double beta[3];
        for (int a = 0; a < 3; ++a) beta[a] = host::kb_beta(J, (double)p->K[a] / (double)p->N[a]);
        auto pad = [](const double (&w)[kJ], int o, float* out8) {
            for (int i = 0; i < 8; ++i) out8[i] = (i - o >= 0 && i - o < kJ) ? (float)w[i - o] : 0.f;
        };
        for (int64_t i = 0; i < M; ++i) {
            const int64_t m = perm[i];
            float* r = &recs[(size_t)i * kW3Rec];
            int c[3];
            for (int a = 0; a < 3; ++a) c[a] = (int)((kpack[m] >> (10 * a)) & 1023u) % p->tile[a];
            const int b0 = w3_block_base(c[0]), b1 = w3_block_base(c[1]), zb = c[2] >> 1;
            double w[kJ];
            float tmp[8];
            for (int a = 0; a < 3; ++a) {
                if (p->minmax) p->mm[a].weights(delta64[(size_t)a * M + m], w);
                else host::kb_weights_f64(delta64[(size_t)a * M + m], J, beta[a], w);
                if (a == 0) pad(w, c[0] - b0, r);
                else if (a == 1) pad(w, c[1] - b1, r + 8);
                else {
                    pad(w, c[2] & 1, tmp);
                    for (int pr = 0; pr < 4; ++pr) {          // rotated by the base pair: slot (zb + pr) & 3 holds pair pr
                        r[16 + 2 * ((zb + pr) & 3)] = tmp[2 * pr];
                        r[16 + 2 * ((zb + pr) & 3) + 1] = tmp[2 * pr + 1];
                    }
                }
            }
            const int32_t key = ((b0 * k3Plane + b1 * k3Pitch) << 4) | zb, mi = (int32_t)m;
            std::memcpy(&r[24], &key, 4);
            std::memcpy(&r[25], &mi, 4);
        }
        NU_TRY(dev_upload(&p->d_w3rec, recs, &p->bytes_plan));
    }
    // V^H work items: (tile, sample range), hot tiles split into chunks of at most max_subtile samples
    {
        // default: enough work items to fill the machine at this plan's batch size (148 SMs x ~16 resident warps), but
        // at least 128 samples per item so that the tile flush stays a small share
        int cap = p->opts.max_subtile;
        if (cap <= 0) {
            const int64_t fill = M * (int64_t)p->max_batch / (148 * 16);
            // 3-D: every item stages / flushes a 32-KB tile; measured on config 4 (fill = 886): caps of 512 / 1024 / 1536 / 3072 /
            // 4096 / 8192 give V^H 0.316 / 0.309 / 0.306 / 0.308 / 0.326 / 0.566 ms and V 0.2135 / 0.210 / 0.209 / 0.208 / 0.207 / 0.249 ms
            cap = (d == 2) ? (int)std::max<int64_t>(128, std::min<int64_t>(1024, fill))
                           : (int)std::max<int64_t>(512, std::min<int64_t>(2048, 2 * fill));
        }
        std::vector<WorkItem> items;
        std::vector<int32_t> tstart(p->n_tiles + 1, 0);
        for (int64_t t = 0; t < p->n_tiles; ++t) {
            tstart[t] = (int32_t)items.size();
            const int64_t b = start[t], e = start[t + 1];
            if (e == b) continue;
            int tc[3];
            int64_t r = t;
            for (int a = d - 1; a >= 0; --a) { tc[a] = (int)(r % p->ntile[a]); r /= p->ntile[a]; }
            uint32_t origin = 0;
            for (int a = 0; a < d; ++a) origin |= (uint32_t)(tc[a] * p->tile[a]) << (10 * a);
            const int64_t nchunk = (e - b + cap - 1) / cap;
            for (int64_t c = 0; c < nchunk; ++c) {
                WorkItem w;
                w.origin = origin;
                w.s_begin = (int32_t)(b + (e - b) * c / nchunk);
                w.s_end = (int32_t)(b + (e - b) * (c + 1) / nchunk);
                w.slab = (int32_t)items.size();
                items.push_back(w);
            }
        }
        tstart[p->n_tiles] = (int32_t)items.size();
        p->n_items = (int)items.size();
        p->n_work = p->n_items;
        // longest first: CTAs that start late get the short items
        std::stable_sort(items.begin(), items.end(), [](const WorkItem& a, const WorkItem& b) {
            return (a.s_end - a.s_begin) > (b.s_end - b.s_begin);
        });
        NU_TRY(dev_upload(&p->d_items, items, &p->bytes_plan));
        NU_TRY(dev_upload(&p->d_tile_item_start, tstart, &p->bytes_plan));
    }
    if (p->il_ok) NU_TRY(plan_build_il(p, kpack, delta, delta64));
    // workspace (batch_pad = max_batch, or whole groups of 32 for the interleaved layout); zeroed once so that the idle
    // lanes of a partly filled group hold finite values
    NU_TRY(dev_alloc((void**)&p->d_grid, (size_t)p->batch_pad * p->cells * sizeof(float2), &p->bytes_work));
    CU_TRY(cudaMemset(p->d_grid, 0, (size_t)p->batch_pad * p->cells * sizeof(float2)));
    NU_TRY(dev_alloc((void**)&p->d_ywork, (size_t)p->batch_pad * std::max<int64_t>(M, 1) * sizeof(float2), &p->bytes_work));
    NU_TRY(dev_alloc((void**)&p->d_scal, sizeof(CgScalars), &p->bytes_work));
    return NUFFT_OK;
}

// ------------------------------------------------------------------------------------------------------------
// nufft_adjoint_noalloc: the workspace grid as a file-scope device array (include/nufft.h).  In host code the NAME of a
// __device__ variable is a host-side stand-in, not a device address: the address a kernel can use comes from
// cudaGetSymbolAddress, asked once per device with that device current (every device that loads this module holds its
// own copy of the array).
// ------------------------------------------------------------------------------------------------------------
static __device__ __align__(256) float2 g_noalloc_grid[NUFFT_NOALLOC_MAX_CELLS];
// device ordinal -> address (null: the lookup failed; the entry point then returns NUFFT_ESTATE).  Called under the
// per-device configuration mutex of nufft_plan.
static float2* noalloc_grid_of_device(int dev) {
    static std::vector<std::pair<int, float2*>> known;
    for (const auto& k : known) if (k.first == dev) return k.second;
    float2* ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g_noalloc_grid);
    if (e != cudaSuccess) { g_last_cuda_error = (int)e; (void)cudaGetLastError(); ptr = nullptr; }
    known.emplace_back(dev, ptr);
    return ptr;
}

extern "C" int nufft_plan(int d, const int64_t* Nd, const int64_t* Kd, const int* Jd, int64_t M, const double* om,
                          int max_batch, const nufft_opts* opts, nufft_plan_t* out) {
    if (out) *out = nullptr;
    if (!out || !Nd || !Kd || !Jd || (d < 1 || d > 3) || M < 0 || (M > 0 && !om) || max_batch < 1) return NUFFT_EINVAL;
    if (M > (int64_t)0x7fffffff) return NUFFT_EINVAL;
    for (int a = 0; a < d; ++a) {
        if (Jd[a] != Jd[0] || Jd[a] < kJmin || Jd[a] > kJmax || Jd[a] > Kd[a] || !supported_K(Kd[a])) return NUFFT_EINVAL;
        if (Nd[a] < 2 || (Nd[a] & 1) || Nd[a] >= Kd[a]) return NUFFT_EINVAL;       // any even N < K, per axis
    }
    bool generic_sigma = false;
    for (int a = 0; a < d; ++a) generic_sigma = generic_sigma || Kd[a] != 2 * Nd[a];
    if (opts && (opts->coef_mode < 0 || opts->coef_mode > 1 || opts->adjoint_mode < 0 || opts->adjoint_mode > 2 || opts->interp_mode < 0 ||
                 opts->interp_mode > 3 || opts->batch_layout < 0 || opts->batch_layout > 2 || opts->kernel < 0 ||
                 opts->kernel > 1))
        return NUFFT_EINVAL;
    const bool generic_j = Jd[0] != kJ || (opts && opts->interp_mode == 2);
    // 1-D and the generic-width path have the atomic V^H only
    if ((d == 1 || generic_j) && opts && opts->adjoint_mode == 1) return NUFFT_EINVAL;
    // the dynamic shared-memory opt-ins are per DEVICE: configure once per device ordinal; the plan remembers its device
    int dev = -1;
    CU_TRY(cudaGetDevice(&dev));
    {
        static std::mutex mu;
        static std::vector<int> done;       // device ordinals already configured
        std::lock_guard<std::mutex> lk(mu);
        if (std::find(done.begin(), done.end(), dev) == done.end()) {
            const cudaError_t cfg = configure_all();
            if (cfg != cudaSuccess) { g_last_cuda_error = (int)cfg; (void)cudaGetLastError(); return NUFFT_ECUDA; }
            done.push_back(dev);
        }
    }
    float2* noalloc_grid = nullptr;
    {
        static std::mutex mu_na;
        std::lock_guard<std::mutex> lk(mu_na);
        noalloc_grid = noalloc_grid_of_device(dev);
    }
    nufft_plan_t p = new (std::nothrow) nufft_plan_s();
    if (!p) return NUFFT_ENOMEM;
    p->device = dev;
    p->noalloc_grid = noalloc_grid;
    p->d = d;
    p->M = M;
    p->max_batch = max_batch;
    if (opts) p->opts = *opts;
    p->il_min_batch = (p->opts.batch_layout == 2) ? 2 : kIlMinBatch;
    p->J = Jd[0];
    p->generic_j = generic_j;
    p->minmax = p->opts.kernel == 1;
    p->generic_sigma = generic_sigma;
    p->il_ok = (d == 2) && !generic_j && !generic_sigma && max_batch >= p->il_min_batch && p->opts.batch_layout != 1 && Kd[1] >= 2 * kBandW;
    p->batch_pad = p->il_ok ? ((max_batch + kIL - 1) / kIL) * kIL : max_batch;
    p->nimg = 1; p->cells = 1;
    for (int a = 0; a < d; ++a) {
        p->N[a] = (int)Nd[a]; p->K[a] = (int)Kd[a];
        p->nimg *= Nd[a]; p->cells *= Kd[a];
    }
    int rc = NUFFT_OK;
    try {
        if (M > 0) p->om_host.assign(om, om + (size_t)M * d);
        rc = plan_build(p, om);
    } catch (const std::bad_alloc&) {
        rc = NUFFT_ENOMEM;
    }
    if (rc != NUFFT_OK) { nufft_destroy(p); return rc; }
    *out = p;
    return NUFFT_OK;
}

static void prof_drain(nufft_plan_t p);
extern "C" int nufft_destroy(nufft_plan_t p) {
    if (!p) return NUFFT_EINVAL;
    prof_drain(p);
    for (int a = 0; a < 3; ++a) { cudaFree(p->d_scale[a]); cudaFree(p->d_tw[a]); }
    cudaFree(p->d_kpack); cudaFree(p->d_delta); cudaFree(p->d_perm);
    cudaFree(p->d_grid); cudaFree(p->d_ywork); cudaFree(p->d_imgwork); cudaFree(p->d_solver);
    cudaFree(p->d_scal); cudaFree(p->d_hist);
    cudaFree(p->d_items); cudaFree(p->d_tile_item_start); cudaFree(p->d_slabs);
    for (int a = 0; a < 3; ++a) cudaFree(p->d_sinv[a]);
    cudaFree(p->d_kspace);
    cudaFree(p->d_ones); cudaFree(p->d_that); cudaFree(p->d_dcf_img); cudaFree(p->d_dcf_t);
    cudaFree(p->d_il_kpack); cudaFree(p->d_il_delta); cudaFree(p->d_il_pos); cudaFree(p->d_il_wtab);
    cudaFree(p->d_il_kpack_c); cudaFree(p->d_il_delta_c); cudaFree(p->d_il_gbase); cudaFree(p->d_il_gbase_c); cudaFree(p->d_w3rec); cudaFree(p->d_il_wv); cudaFree(p->d_il_wv_c);
    cudaFree(p->d_il_rowptr); cudaFree(p->d_il_v2h); cudaFree(p->d_il_items); cudaFree(p->d_yil);
    cudaFree(p->d_il_kpack_t); cudaFree(p->d_il_delta_t); cudaFree(p->d_il_gbase_t); cudaFree(p->d_il_wv_t); cudaFree(p->d_il_t2h); cudaFree(p->d_il_titems);
    if (p->cg_graph) cudaGraphExecDestroy(p->cg_graph);
    for (auto& og : p->op_graphs) cudaGraphExecDestroy(og.exec);
    if (p->hp_h2d) cudaStreamDestroy(p->hp_h2d);
    if (p->hp_d2h) cudaStreamDestroy(p->hp_d2h);
    for (int i = 0; i < 2; ++i) {
        if (p->hp_in[i]) cudaEventDestroy(p->hp_in[i]);
        if (p->hp_cmp[i]) cudaEventDestroy(p->hp_cmp[i]);
        if (p->hp_out[i]) cudaEventDestroy(p->hp_out[i]);
        cudaFree(p->hp_din[i]); cudaFree(p->hp_dout[i]);
    }
    if (p->hp_start) cudaEventDestroy(p->hp_start);
    (void)cudaGetLastError();
    delete p;
    return NUFFT_OK;
}

extern "C" int nufft_plan_info(nufft_plan_t p, int64_t* bytes_plan, int64_t* bytes_work, int64_t* n_tiles,
                               int64_t* n_work, int64_t* max_tile_samples) {
    if (!p) return NUFFT_EINVAL;
    if (bytes_plan) *bytes_plan = p->bytes_plan;
    if (bytes_work) *bytes_work = p->bytes_work;
    if (n_tiles) *n_tiles = p->n_tiles;
    if (n_work) *n_work = p->n_work;
    if (max_tile_samples) *max_tile_samples = p->max_tile_samples;
    return NUFFT_OK;
}

extern "C" int nufft_plan_tile_histogram(nufft_plan_t p, int64_t* counts) {
    if (!p || !counts) return NUFFT_EINVAL;
    for (int k = 0; k < NUFFT_TILE_HIST_BUCKETS; ++k) counts[k] = p->tile_hist[k];
    return NUFFT_OK;
}

extern "C" int nufft_plan_modes(nufft_plan_t p, int* J, int* kernel, int* paths, double* poly_err) {
    if (!p) return NUFFT_EINVAL;
    if (J) *J = p->J;
    if (kernel) *kernel = p->minmax ? 1 : 0;
    if (paths) *paths = (p->il_ok ? 1 : 0) | (p->il_ok && p->il_coherent ? 2 : 0) | (p->generic_j ? 4 : 0) | (p->toep_on ? 8 : 0);
    if (poly_err) *poly_err = p->poly_err;
    return NUFFT_OK;
}

extern "C" int64_t nufft_launch_count(nufft_plan_t p) { return p ? p->launches : -1; }

static void prof_drain(nufft_plan_t p) {
    for (auto& r : p->prof) {
        if (cudaEventSynchronize(r.b) == cudaSuccess) {
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, r.a, r.b) == cudaSuccess) { p->prof_ms[r.label] += ms; p->prof_n[r.label]++; }
        }
        cudaEventDestroy(r.a);
        cudaEventDestroy(r.b);
    }
    (void)cudaGetLastError();
    p->prof.clear();
}
extern "C" int nufft_profile_enable(nufft_plan_t p, int on) {
    if (!p) return NUFFT_EINVAL;
    p->prof_on = on != 0;
    return NUFFT_OK;
}
extern "C" int nufft_profile_reset(nufft_plan_t p) {
    if (!p) return NUFFT_EINVAL;
    prof_drain(p);
    std::fill(p->prof_ms.begin(), p->prof_ms.end(), 0.0);
    std::fill(p->prof_n.begin(), p->prof_n.end(), 0);
    return NUFFT_OK;
}
extern "C" int nufft_profile_count(nufft_plan_t p) {
    if (!p) return NUFFT_EINVAL;
    return (int)p->prof_labels.size();
}
extern "C" int nufft_profile_get(nufft_plan_t p, int i, const char** name, double* total_ms, int64_t* launches) {
    if (!p || i < 0 || i >= (int)p->prof_labels.size()) return NUFFT_EINVAL;
    prof_drain(p);
    if (name) *name = p->prof_labels[i];
    if (total_ms) *total_ms = p->prof_ms[i];
    if (launches) *launches = p->prof_n[i];
    return NUFFT_OK;
}

// ------------------------------------------------------------------------------------------------------------
// transforms
// ------------------------------------------------------------------------------------------------------------
static bool wrong_device(nufft_plan_t p) {
    int dev = -1;
    return cudaGetDevice(&dev) != cudaSuccess || dev != p->device;
}
// every transform / solver entry point goes through this: null plan, batch out of range, or a current device other than the
// plan's (its buffers and kernel attributes belong to that device) -> NUFFT_EINVAL
static bool bad_batch(nufft_plan_t p, int batch) { return !p || batch < 1 || batch > p->max_batch || wrong_device(p); }

extern "C" int nufft_stage_scale_fft(nufft_plan_t p, int batch, const nufft_c64* x, nufft_c64* grid, void* stream) {
    if (bad_batch(p, batch) || !x || !grid) return NUFFT_EINVAL;
    return run_scale_fft(p, batch, (const float2*)x, (float2*)grid, nullptr, false, (cudaStream_t)stream);
}
extern "C" int nufft_stage_interp(nufft_plan_t p, int batch, const nufft_c64* grid, nufft_c64* y, void* stream) {
    if (bad_batch(p, batch) || !grid || (!y && p->M > 0)) return NUFFT_EINVAL;
    return run_interp(p, batch, (const float2*)grid, (float2*)y, (cudaStream_t)stream);
}
extern "C" int nufft_stage_gridding(nufft_plan_t p, int batch, const nufft_c64* y, nufft_c64* grid, void* stream) {
    if (bad_batch(p, batch) || !grid || (!y && p->M > 0)) return NUFFT_EINVAL;
    return run_gridding(p, batch, (const float2*)y, (float2*)grid, (cudaStream_t)stream);
}
extern "C" int nufft_stage_fft_scale(nufft_plan_t p, int batch, nufft_c64* grid, nufft_c64* x, void* stream) {
    if (bad_batch(p, batch) || !x || !grid) return NUFFT_EINVAL;
    return run_fft_scale(p, batch, (float2*)grid, (float2*)x, nullptr, (cudaStream_t)stream);
}

static int forward_impl(nufft_plan_t p, int batch, const nufft_c64* x, nufft_c64* y, cudaStream_t st) {
    if (use_il(p, batch)) {
        NU_TRY(run_scale_fft_il(p, batch, (const float2*)x, p->d_grid, nullptr, false, st));
        if (p->il_coherent) return run_interp_il_caller(p, batch, p->d_grid, (float2*)y, st);
        NU_TRY(run_interp_il(p, batch, p->d_grid, p->d_ywork, st));
        return run_y_from_il(p, batch, p->d_ywork, (float2*)y, st);
    }
    NU_TRY(run_scale_fft(p, batch, (const float2*)x, p->d_grid, nullptr, false, st));
    return run_interp(p, batch, p->d_grid, (float2*)y, st);
}

static int adjoint_impl(nufft_plan_t p, int batch, const nufft_c64* y, nufft_c64* x, cudaStream_t st) {
    if (use_il(p, batch)) {
        NU_TRY(run_y_to_il(p, batch, (const float2*)y, st));
        NU_TRY(run_gridding_il(p, batch, p->d_yil, p->d_grid, st));
        return run_fft_scale_il(p, batch, p->d_grid, (float2*)x, nullptr, st);
    }
    NU_TRY(run_gridding(p, batch, (const float2*)y, p->d_grid, st));
    return run_fft_scale(p, batch, p->d_grid, (float2*)x, nullptr, st);
}

static int selfadjoint_impl(nufft_plan_t p, int batch, const nufft_c64* x_in, nufft_c64* x_out, cudaStream_t st) {
    if (use_il(p, batch)) {     // the intermediate samples stay sorted and interleaved: no scatter, no gather
        NU_TRY(run_scale_fft_il(p, batch, (const float2*)x_in, p->d_grid, nullptr, false, st));
        NU_TRY(run_interp_il(p, batch, p->d_grid, p->d_ywork, st));
        NU_TRY(run_gridding_il(p, batch, p->d_ywork, p->d_grid, st));
        return run_fft_scale_il(p, batch, p->d_grid, (float2*)x_out, nullptr, st);
    }
    NU_TRY(run_scale_fft(p, batch, (const float2*)x_in, p->d_grid, nullptr, false, st));
    NU_TRY(run_interp(p, batch, p->d_grid, p->d_ywork, st));
    NU_TRY(run_gridding(p, batch, p->d_ywork, p->d_grid, st));
    return run_fft_scale(p, batch, p->d_grid, (float2*)x_out, nullptr, st);
}

// opts.use_graphs: a transform call whose (kind, batch, pointers, stream) was seen before is replayed as one CUDA graph
// (solver loops and the host pipeline call with fixed pointers; single small transforms are launch-latency bound).  The
// first call of each kind and layout runs eagerly so that lazy allocations happen outside a capture; calls made while the
// stream is already capturing (the CG iteration graph) and calls on the legacy stream run eagerly.
template <class F>
static int run_graphed(nufft_plan_t p, int kind, int batch, const void* in, void* out, cudaStream_t st, F impl) {
    const int il = use_il(p, batch) ? 1 : 0;
    bool eager = !p->opts.use_graphs || p->prof_on || st == nullptr || !p->op_warm[kind][il];
    if (!eager) {
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(st, &cs) != cudaSuccess || cs != cudaStreamCaptureStatusNone) eager = true;
    }
    if (eager) {
        const int rc = impl();
        if (rc == NUFFT_OK) p->op_warm[kind][il] = true;
        return rc;
    }
    for (auto& g : p->op_graphs)
        if (g.kind == kind && g.batch == batch && g.in == in && g.out == out && g.stream == (void*)st) {
            CU_TRY(cudaGraphLaunch(g.exec, st));
            p->launches += g.launches;
            return NUFFT_OK;
        }
    const int64_t l0 = p->launches;
    CU_TRY(cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal));
    const int rc = impl();
    cudaGraph_t g = nullptr;
    const cudaError_t e = cudaStreamEndCapture(st, &g);
    const int nl = (int)(p->launches - l0);
    p->launches = l0;
    if (rc != NUFFT_OK || e != cudaSuccess || !g) {
        if (g) cudaGraphDestroy(g);
        (void)cudaGetLastError();
        if (rc != NUFFT_OK) return rc;
        g_last_cuda_error = (int)e;
        return NUFFT_ECUDA;
    }
    nufft_plan_s::OpGraph og{kind, batch, in, out, (void*)st, nullptr, nl};
    const cudaError_t ei = cudaGraphInstantiate(&og.exec, g, 0);
    cudaGraphDestroy(g);
    if (ei != cudaSuccess) { g_last_cuda_error = (int)ei; (void)cudaGetLastError(); return NUFFT_ECUDA; }
    if (p->op_graphs.size() >= 16) {            // small FIFO cache
        cudaGraphExecDestroy(p->op_graphs.front().exec);
        p->op_graphs.erase(p->op_graphs.begin());
    }
    p->op_graphs.push_back(og);
    CU_TRY(cudaGraphLaunch(og.exec, st));
    p->launches += nl;
    return NUFFT_OK;
}

extern "C" int nufft_forward(nufft_plan_t p, int batch, const nufft_c64* x, nufft_c64* y, void* stream) {
    if (bad_batch(p, batch) || !x || (!y && p->M > 0)) return NUFFT_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    return run_graphed(p, 0, batch, x, y, st, [&]() { return forward_impl(p, batch, x, y, st); });
}
extern "C" int nufft_adjoint(nufft_plan_t p, int batch, const nufft_c64* y, nufft_c64* x, void* stream) {
    if (bad_batch(p, batch) || !x || (!y && p->M > 0)) return NUFFT_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    return run_graphed(p, 1, batch, y, x, st, [&]() { return adjoint_impl(p, batch, y, x, st); });
}
// x = A^H y, one image, with the workspace grid in the library's static device array: no allocation of any kind on this path
// (run_gridding zero-fills the cells it accumulates into; adjoint_mode = 1 would allocate its slabs on first use and the
// profiler creates events, so both are refused).
extern "C" int nufft_adjoint_noalloc(nufft_plan_t p, const nufft_c64* y, nufft_c64* x, void* stream) {
    if (bad_batch(p, 1) || !x || (!y && p->M > 0)) return NUFFT_EINVAL;
    if (p->cells > (int64_t)NUFFT_NOALLOC_MAX_CELLS) return NUFFT_ETOOBIG;
    if (p->opts.adjoint_mode == 1 || p->prof_on) return NUFFT_EINVAL;
    if (!p->noalloc_grid) return NUFFT_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    NU_TRY(run_gridding(p, 1, (const float2*)y, p->noalloc_grid, st));
    return run_fft_scale(p, 1, p->noalloc_grid, (float2*)x, nullptr, st);
}
extern "C" int nufft_selfadjoint(nufft_plan_t p, int batch, const nufft_c64* x_in, nufft_c64* x_out, void* stream) {
    if (bad_batch(p, batch) || !x_in || !x_out) return NUFFT_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    return run_graphed(p, 2, batch, x_in, x_out, st, [&]() { return selfadjoint_impl(p, batch, x_in, x_out, st); });
}

// ------------------------------------------------------------------------------------------------------------
// host-buffer transforms: chunked pipeline  H2D (copy stream) -> kernels (caller's stream) -> D2H (second copy stream)
// ------------------------------------------------------------------------------------------------------------
static int host_pipe_init(nufft_plan_t p) {
    if (p->hp_ready) return NUFFT_OK;
    CU_TRY(cudaStreamCreateWithFlags(&p->hp_h2d, cudaStreamNonBlocking));
    CU_TRY(cudaStreamCreateWithFlags(&p->hp_d2h, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) {
        CU_TRY(cudaEventCreateWithFlags(&p->hp_in[i], cudaEventDisableTiming));
        CU_TRY(cudaEventCreateWithFlags(&p->hp_cmp[i], cudaEventDisableTiming));
        CU_TRY(cudaEventCreateWithFlags(&p->hp_out[i], cudaEventDisableTiming));
    }
    CU_TRY(cudaEventCreateWithFlags(&p->hp_start, cudaEventDisableTiming));
    p->hp_chunk = std::min(p->max_batch, p->il_ok ? kIL : 8);
    const size_t per = (size_t)std::max<int64_t>(p->nimg, std::max<int64_t>(p->M, 1)) * sizeof(float2);
    for (int i = 0; i < 2; ++i) {
        NU_TRY(dev_alloc((void**)&p->hp_din[i], (size_t)p->hp_chunk * per, &p->bytes_work));
        NU_TRY(dev_alloc((void**)&p->hp_dout[i], (size_t)p->hp_chunk * per, &p->bytes_work));
    }
    p->hp_ready = true;
    return NUFFT_OK;
}

// kind: 0 = forward (in: images, out: samples), 1 = adjoint (in: samples, out: images), 2 = selfadjoint (images both)
static int host_pipeline(nufft_plan_t p, int kind, int batch, const nufft_c64* in_host, nufft_c64* out_host,
                         cudaStream_t st) {
    NU_TRY(host_pipe_init(p));
    const int64_t n_in = (kind == 1) ? p->M : p->nimg, n_out = (kind == 0) ? p->M : p->nimg;
    const int CH = p->hp_chunk;
    CU_TRY(cudaEventRecord(p->hp_start, st));
    // strict mode: the copies in are ordered after everything already enqueued on the caller's stream.  With
    // nufft_host_input_ready(p, 1) the caller promises that the host input is final when the call is made, so the
    // first copy in may overlap the copy back of the previous call (only the staging buffers are waited for).
    if (!p->hp_input_ready) CU_TRY(cudaStreamWaitEvent(p->hp_h2d, p->hp_start, 0));
    CU_TRY(cudaStreamWaitEvent(p->hp_d2h, p->hp_start, 0));
    // Interleaved path: the kernels of a chunk cost the same for 16 and for 32 images (lanes = images), the copies do not,
    // and the pipeline is copy-bound: chunks of 16 images start the first kernels and the first copy back earlier
    // (cfg2 batch 64, strict order: 1.165 -> 1.047 ms per A^H A).  A remainder of fewer than kIlMinBatch images is merged
    // into the last chunk so that no chunk falls back to the planar path.
    // (With nufft_host_input_ready the calls overlap one another and the steady state is bound by the copies alone: full
    // 32-image chunks then keep the kernel time per image lowest -- 73.6 k against 71.9 k pairs/s.)
    const int step = (p->il_ok && CH == kIL && batch >= 2 * kIlMinBatch && !p->hp_input_ready) ? kIL / 2 : CH;
    int c = 0;
    for (int b0 = 0, n = 0; b0 < batch; b0 += n, ++c) {
        n = std::min(step, batch - b0);
        if (step < CH && batch - b0 - n > 0 && batch - b0 - n < kIlMinBatch && batch - b0 <= CH) n = batch - b0;
        const int buf = c & 1;
        if (c >= 2 || p->hp_used[buf]) CU_TRY(cudaStreamWaitEvent(p->hp_h2d, p->hp_cmp[buf], 0));   // last reader of din[buf]
        if (n_in > 0)
            CU_TRY(cudaMemcpyAsync(p->hp_din[buf], (const float2*)in_host + (int64_t)b0 * n_in,
                                   (size_t)n * n_in * sizeof(float2), cudaMemcpyHostToDevice, p->hp_h2d));
        CU_TRY(cudaEventRecord(p->hp_in[buf], p->hp_h2d));
        CU_TRY(cudaStreamWaitEvent(st, p->hp_in[buf], 0));
        if (c >= 2) CU_TRY(cudaStreamWaitEvent(st, p->hp_out[buf], 0));             // D2H of chunk c-2 has read dout[buf]
        int rc;
        if (kind == 0) rc = nufft_forward(p, n, (const nufft_c64*)p->hp_din[buf], (nufft_c64*)p->hp_dout[buf], st);
        else if (kind == 1) rc = nufft_adjoint(p, n, (const nufft_c64*)p->hp_din[buf], (nufft_c64*)p->hp_dout[buf], st);
        else rc = nufft_selfadjoint(p, n, (const nufft_c64*)p->hp_din[buf], (nufft_c64*)p->hp_dout[buf], st);
        NU_TRY(rc);
        CU_TRY(cudaEventRecord(p->hp_cmp[buf], st));
        p->hp_used[buf] = true;
        CU_TRY(cudaStreamWaitEvent(p->hp_d2h, p->hp_cmp[buf], 0));
        if (n_out > 0)
            CU_TRY(cudaMemcpyAsync((float2*)out_host + (int64_t)b0 * n_out, p->hp_dout[buf],
                                   (size_t)n * n_out * sizeof(float2), cudaMemcpyDeviceToHost, p->hp_d2h));
        CU_TRY(cudaEventRecord(p->hp_out[buf], p->hp_d2h));
    }
    // join: the caller's stream continues only after the last copies back
    CU_TRY(cudaStreamWaitEvent(st, p->hp_out[0], 0));
    if (c >= 2) CU_TRY(cudaStreamWaitEvent(st, p->hp_out[1], 0));
    return NUFFT_OK;
}

extern "C" int nufft_host_input_ready(nufft_plan_t p, int on) {
    if (!p) return NUFFT_EINVAL;
    p->hp_input_ready = on != 0;
    return NUFFT_OK;
}
extern "C" int nufft_forward_host(nufft_plan_t p, int batch, const nufft_c64* x_host, nufft_c64* y_host, void* stream) {
    if (bad_batch(p, batch) || !x_host || (!y_host && p->M > 0)) return NUFFT_EINVAL;
    return host_pipeline(p, 0, batch, x_host, y_host, (cudaStream_t)stream);
}
extern "C" int nufft_adjoint_host(nufft_plan_t p, int batch, const nufft_c64* y_host, nufft_c64* x_host, void* stream) {
    if (bad_batch(p, batch) || !x_host || (!y_host && p->M > 0)) return NUFFT_EINVAL;
    return host_pipeline(p, 1, batch, y_host, x_host, (cudaStream_t)stream);
}
extern "C" int nufft_selfadjoint_host(nufft_plan_t p, int batch, const nufft_c64* x_in_host, nufft_c64* x_out_host,
                                      void* stream) {
    if (bad_batch(p, batch) || !x_in_host || !x_out_host) return NUFFT_EINVAL;
    return host_pipeline(p, 2, batch, x_in_host, x_out_host, (cudaStream_t)stream);
}

// ------------------------------------------------------------------------------------------------------------
// multi-coil operator, eqs. (34)-(35)
// ------------------------------------------------------------------------------------------------------------
extern "C" int nufft_set_coils(nufft_plan_t p, int ncoil, const nufft_c64* c) {
    if (!p || wrong_device(p) || ncoil < 0 || ncoil > p->max_batch || (ncoil > 0 && !c)) return NUFFT_EINVAL;
    p->ncoil = ncoil;
    p->d_coils = (ncoil > 0) ? (const float2*)c : nullptr;
    if (p->cg_graph) { cudaGraphExecDestroy(p->cg_graph); p->cg_graph = nullptr; }   // the coil pointer is baked into it
    if (ncoil > 0 && !p->d_imgwork)
        NU_TRY(dev_alloc((void**)&p->d_imgwork, (size_t)p->max_batch * p->nimg * sizeof(float2), &p->bytes_work));
    return NUFFT_OK;
}

static int coil_reduce(nufft_plan_t p, float2* x, cudaStream_t st) {
    const int blocks = (int)std::min<int64_t>((p->nimg + 255) / 256, 148 * 8);
    coil_sum_kernel<<<blocks, 256, 0, st>>>(x, p->d_imgwork, p->ncoil, p->nimg);
    CU_TRY(cudaGetLastError());
    p->launches++;
    return NUFFT_OK;
}

extern "C" int nufft_forward_coils(nufft_plan_t p, const nufft_c64* x, nufft_c64* y, void* stream) {
    if (!p || wrong_device(p) || !x || (!y && p->M > 0)) return NUFFT_EINVAL;
    if (p->ncoil < 1) return NUFFT_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    if (use_il(p, p->ncoil)) {
        NU_TRY(run_scale_fft_il(p, p->ncoil, (const float2*)x, p->d_grid, p->d_coils, true, st));
        if (p->il_coherent) return run_interp_il_caller(p, p->ncoil, p->d_grid, (float2*)y, st);
        NU_TRY(run_interp_il(p, p->ncoil, p->d_grid, p->d_ywork, st));
        return run_y_from_il(p, p->ncoil, p->d_ywork, (float2*)y, st);
    }
    NU_TRY(run_scale_fft(p, p->ncoil, (const float2*)x, p->d_grid, p->d_coils, true, st));
    return run_interp(p, p->ncoil, p->d_grid, (float2*)y, st);
}

extern "C" int nufft_adjoint_coils(nufft_plan_t p, const nufft_c64* y, nufft_c64* x, void* stream) {
    if (!p || wrong_device(p) || !x || (!y && p->M > 0)) return NUFFT_EINVAL;
    if (p->ncoil < 1) return NUFFT_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    if (use_il(p, p->ncoil)) {
        NU_TRY(run_y_to_il(p, p->ncoil, (const float2*)y, st));
        NU_TRY(run_gridding_il(p, p->ncoil, p->d_yil, p->d_grid, st));
        return run_fft_scale_il(p, p->ncoil, p->d_grid, (float2*)x, p->d_coils, st, true);
    }
    NU_TRY(run_gridding(p, p->ncoil, (const float2*)y, p->d_grid, st));
    NU_TRY(run_fft_scale(p, p->ncoil, p->d_grid, p->d_imgwork, p->d_coils, st));
    return coil_reduce(p, (float2*)x, st);
}

extern "C" int nufft_selfadjoint_coils(nufft_plan_t p, const nufft_c64* x_in, nufft_c64* x_out, void* stream) {
    if (!p || wrong_device(p) || !x_in || !x_out) return NUFFT_EINVAL;
    if (p->ncoil < 1) return NUFFT_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    if (use_il(p, p->ncoil)) {
        NU_TRY(run_scale_fft_il(p, p->ncoil, (const float2*)x_in, p->d_grid, p->d_coils, true, st));
        NU_TRY(run_interp_il(p, p->ncoil, p->d_grid, p->d_ywork, st));
        NU_TRY(run_gridding_il(p, p->ncoil, p->d_ywork, p->d_grid, st));
        return run_fft_scale_il(p, p->ncoil, p->d_grid, (float2*)x_out, p->d_coils, st, true);
    }
    NU_TRY(run_scale_fft(p, p->ncoil, (const float2*)x_in, p->d_grid, p->d_coils, true, st));
    NU_TRY(run_interp(p, p->ncoil, p->d_grid, p->d_ywork, st));
    NU_TRY(run_gridding(p, p->ncoil, p->d_ywork, p->d_grid, st));
    NU_TRY(run_fft_scale(p, p->ncoil, p->d_grid, p->d_imgwork, p->d_coils, st));
    return coil_reduce(p, (float2*)x_out, st);
}

// ------------------------------------------------------------------------------------------------------------
// "next" rows of SURVEY 8(f): density compensation (eqs. 6-7) and Toeplitz A^H A
// ------------------------------------------------------------------------------------------------------------
static int ew_blocks(int64_t n);

extern "C" int nufft_density_weights(nufft_plan_t p, int niter, nufft_c64* w, void* stream) {
    if (!p || wrong_device(p) || niter < 0 || (!w && p->M > 0)) return NUFFT_EINVAL;
    if (p->M == 0) return NUFFT_OK;
    cudaStream_t st = (cudaStream_t)stream;
    if (!p->d_dcf_img) NU_TRY(dev_alloc((void**)&p->d_dcf_img, (size_t)p->nimg * sizeof(float2), &p->bytes_work));
    if (!p->d_dcf_t) NU_TRY(dev_alloc((void**)&p->d_dcf_t, (size_t)p->M * sizeof(float2), &p->bytes_work));
    const int nb = ew_blocks(p->M);
    dcf_init_kernel<<<nb, 256, 0, st>>>((float2*)w, p->M);
    p->launches++;
    for (int i = 0; i < niter; ++i) {          // w <- w / |A A^H w|   (eq. 6, R21)
        NU_TRY(nufft_adjoint(p, 1, w, (nufft_c64*)p->d_dcf_img, st));
        NU_TRY(nufft_forward(p, 1, (const nufft_c64*)p->d_dcf_img, (nufft_c64*)p->d_dcf_t, st));
        dcf_update_kernel<<<nb, 256, 0, st>>>((float2*)w, p->d_dcf_t, p->M);
        p->launches++;
    }
    CU_TRY(cudaGetLastError());
    return NUFFT_OK;
}

extern "C" int nufft_adjoint_dcf(nufft_plan_t p, int batch, const nufft_c64* y, const nufft_c64* w, nufft_c64* x,
                                 void* stream) {
    if (bad_batch(p, batch) || !x || ((!y || !w) && p->M > 0)) return NUFFT_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    if (p->M > 0) {       // x = A^H (y . w)   (eq. 7); d_ywork is free during an adjoint
        weight_mul_kernel<<<ew_blocks(p->M * batch), 256, 0, st>>>(p->d_ywork, (const float2*)y, (const float2*)w, p->M, batch);
        CU_TRY(cudaGetLastError());
        p->launches++;
    }
    return nufft_adjoint(p, batch, (const nufft_c64*)p->d_ywork, x, st);
}

template <int K> static void launch_rows_full(float2* data, const float2* tw, int nlines, cudaStream_t st) {
    constexpr int threads = FftGeom<K>::TPL * Rad<K>::LC;
    fft_rows_full_kernel<K><<<(nlines + Rad<K>::LC - 1) / Rad<K>::LC, threads, smem_rows<K>(), st>>>(data, tw, nlines);
}
template <int K> static void launch_cols_full(const ColPassParams& c, cudaStream_t st) {
    constexpr int threads = FftGeom<K>::TPL * Rad<K>::TS;
    fft_cols_kernel<K, false, true><<<c.ngroups, threads, smem_cols<K>(), st>>>(c);
}
#define NUFFT_K_SWITCH(K, CALL)                                                                                \
    switch (K) {                                                                                               \
        case 32: CALL(32); break; case 64: CALL(64); break; case 128: CALL(128); break;                        \
        case 256: CALL(256); break; case 512: CALL(512); break; case 1024: CALL(1024); break;                  \
        default: return NUFFT_EINVAL;                                                                          \
    }

// in-place unpruned forward FFT of a planar K^d array (used once per plan for the Toeplitz spectrum)
static int fft_full_inplace(nufft_plan_t p, float2* data, cudaStream_t st, int batch, bool do_rows) {
    const int d = p->d;
    const int64_t cells = p->cells;
    if (do_rows) {
        const int Kl = p->K[d - 1];
        const int nlines = (int)(cells / Kl) * batch;
#define CALL_ROWS(KK) launch_rows_full<KK>(data, p->d_tw[d - 1], nlines, st)
        NUFFT_K_SWITCH(Kl, CALL_ROWS)
#undef CALL_ROWS
    }
    for (int a = d - 2; a >= 0; --a) {
        ColPassParams c{};
        c.grid = data; c.tw = p->d_tw[a];
        c.batch_stride = cells;
        int64_t inner = 1;
        for (int b = a + 1; b < d; ++b) inner *= p->K[b];
        c.line_stride = inner; c.inner = (int)inner;
        c.n_outer = (a == 0) ? 1 : p->K[0]; c.k_outer = 0;
        c.outer_stride = (a == 0) ? 0 : (int64_t)p->K[1] * p->K[2];
        c.ngroups = batch * c.n_outer * (c.inner / tile_T(p->K[a]));
#define CALL_COLS(KK) launch_cols_full<KK>(c, st)
        NUFFT_K_SWITCH(p->K[a], CALL_COLS)
#undef CALL_COLS
    }
    CU_TRY(cudaGetLastError());
    p->launches += do_rows ? d : d - 1;
    return NUFFT_OK;
}

extern "C" int nufft_toeplitz_build(nufft_plan_t p, const nufft_c64* w, void* stream) {
    if (!p) return NUFFT_EINVAL;
    if (p->generic_sigma) return NUFFT_EINVAL;      // the embedding lives on the K = 2 N grid (reading R22)
    cudaStream_t st = (cudaStream_t)stream;
    const int d = p->d;
    const int64_t M = p->M;
    if (!p->d_that) NU_TRY(dev_alloc((void**)&p->d_that, (size_t)p->cells * sizeof(float2), &p->bytes_plan));
    if (!p->d_dcf_img) NU_TRY(dev_alloc((void**)&p->d_dcf_img, (size_t)p->nimg * sizeof(float2), &p->bytes_work));
    // T[d' + s] = sum_m (w_m e^{i om_m . s}) e^{i om_m . d'}: 2^d adjoint NUFFTs of phase-modulated weights on this plan's own
    // geometry, one per half-shift s in {-N/2, +N/2}^d (R22); the modulation is computed on the host in float64.
    std::vector<float2> wh((size_t)std::max<int64_t>(M, 1), make_float2(1.f, 0.f)), wmod((size_t)std::max<int64_t>(M, 1));
    if (w && M > 0) {
        CU_TRY(cudaMemcpyAsync(wh.data(), w, (size_t)M * sizeof(float2), cudaMemcpyDeviceToHost, st));
        CU_TRY(cudaStreamSynchronize(st));
    }
    float2* d_wmod = nullptr;
    NU_TRY(dev_alloc((void**)&d_wmod, (size_t)std::max<int64_t>(M, 1) * sizeof(float2), nullptr));
    int rc = NUFFT_OK;
    const int nb_img = ew_blocks(p->nimg);
    for (int blk = 0; blk < (1 << d) && rc == NUFFT_OK; ++blk) {
        int h[3] = {0, 0, 0};
        double shift[3] = {0.0, 0.0, 0.0};
        for (int a = 0; a < d; ++a) { h[a] = (blk >> a) & 1; shift[a] = (h[a] - 0.5) * (double)p->N[a]; }
        for (int64_t m = 0; m < M; ++m) {
            double ph = 0.0;
            for (int a = 0; a < d; ++a) ph += p->om_host[(size_t)m * d + a] * shift[a];
            const double c = std::cos(ph), sn = std::sin(ph);
            wmod[m] = make_float2((float)(wh[m].x * c - wh[m].y * sn), (float)(wh[m].x * sn + wh[m].y * c));
        }
        cudaError_t e = cudaMemcpyAsync(d_wmod, wmod.data(), (size_t)std::max<int64_t>(M, 1) * sizeof(float2), cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);          // wmod is reused by the next block
        if (e != cudaSuccess) { g_last_cuda_error = (int)e; rc = NUFFT_ECUDA; break; }
        rc = adjoint_impl(p, 1, (const nufft_c64*)d_wmod, (nufft_c64*)p->d_dcf_img, st);
        if (rc != NUFFT_OK) break;
        psf_place_block_kernel<<<nb_img, 256, 0, st>>>(p->d_that, p->d_dcf_img, p->N[0], p->N[1], p->N[2], h[0], h[1], h[2]);
        p->launches++;
    }
    if (rc == NUFFT_OK) {
        const int nb = ew_blocks(p->cells);
        psf_zero_planes_kernel<<<nb, 256, 0, st>>>(p->d_that, p->K[0], p->K[1], d == 3 ? p->K[2] : 1);
        rc = fft_full_inplace(p, p->d_that, st);
        if (rc == NUFFT_OK) psf_sign_kernel<<<nb, 256, 0, st>>>(p->d_that, p->K[0], p->K[1], d == 3 ? p->K[2] : 1,
                                                                   (float)(1.0 / (double)p->cells));
        p->launches += 2;
    }
    const cudaError_t e = cudaStreamSynchronize(st);
    cudaFree(d_wmod);
    if (rc == NUFFT_OK && e != cudaSuccess) { g_last_cuda_error = (int)e; rc = NUFFT_ECUDA; }
    if (rc == NUFFT_OK && cudaGetLastError() != cudaSuccess) rc = NUFFT_ECUDA;
    return rc;
}

extern "C" int nufft_toeplitz_enable(nufft_plan_t p, int on) {
    if (!p) return NUFFT_EINVAL;
    if (on && !p->d_that) return NUFFT_ESTATE;
    p->toep_on = on != 0;
    return NUFFT_OK;
}

// x_out = crop(F^H(T^ . F(pad x_in))); coils: sum_i conj(c_i) crop(F^H(T^ . F(pad c_i x_in)))
// coil != nullptr on the interleaved path: x_out is the coil-SUMMED image (sum fused into the last pass); on the planar path
// x_out receives the per-coil images and the caller reduces them.  *summed tells which.
static int run_toeplitz(nufft_plan_t p, int batch, const float2* x_in, float2* x_out, float2* x_sum, const float2* coil,
                        bool same_image, cudaStream_t st, bool* summed = nullptr) {
    p->unit_scale = true;
    p->cur_mult = p->d_that;
    int rc;
    if (use_il(p, batch)) {
        rc = run_scale_fft_il(p, batch, x_in, p->d_grid, coil, same_image, st);
        const bool fuse = coil != nullptr && x_sum != nullptr;
        if (rc == NUFFT_OK) rc = run_fft_scale_il(p, batch, p->d_grid, fuse ? x_sum : x_out, coil, st, fuse);
        if (summed) *summed = fuse;
    } else {
        rc = run_scale_fft(p, batch, x_in, p->d_grid, coil, same_image, st);
        if (rc == NUFFT_OK) rc = run_fft_scale(p, batch, p->d_grid, x_out, coil, st);
    }
    p->unit_scale = false;
    p->cur_mult = nullptr;
    return rc;
}

extern "C" int nufft_selfadjoint_toeplitz(nufft_plan_t p, int batch, const nufft_c64* x_in, nufft_c64* x_out, void* stream) {
    if (bad_batch(p, batch) || !x_in || !x_out) return NUFFT_EINVAL;
    if (!p->d_that) return NUFFT_ESTATE;
    return run_toeplitz(p, batch, (const float2*)x_in, (float2*)x_out, nullptr, nullptr, false, (cudaStream_t)stream);
}

// ------------------------------------------------------------------------------------------------------------
// solvers
// ------------------------------------------------------------------------------------------------------------
static int ew_blocks(int64_t n) { return (int)std::max<int64_t>(1, std::min<int64_t>((n + 255) / 256, 148 * 8)); }

static int ensure_solver(nufft_plan_t p, int64_t nvec, int hist) {
    if (p->solver_vecs < nvec) {
        cudaFree(p->d_solver);
        p->d_solver = nullptr;
        p->solver_vecs = 0;
        NU_TRY(dev_alloc((void**)&p->d_solver, (size_t)nvec * p->nimg * sizeof(float2), &p->bytes_work));
        p->solver_vecs = nvec;
    }
    if (p->hist_cap < hist) {
        cudaFree(p->d_hist);
        p->d_hist = nullptr;
        p->hist_cap = 0;
        NU_TRY(dev_alloc((void**)&p->d_hist, (size_t)hist * sizeof(double), &p->bytes_work));
        p->hist_cap = hist;
    }
    return NUFFT_OK;
}

static int coil_reduce(nufft_plan_t p, float2* x, cudaStream_t st);
extern "C" int nufft_selfadjoint_toeplitz_coils(nufft_plan_t p, const nufft_c64* x_in, nufft_c64* x_out, void* stream) {
    if (!p || wrong_device(p) || !x_in || !x_out) return NUFFT_EINVAL;
    if (p->ncoil < 1 || !p->d_that) return NUFFT_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    bool summed = false;
    NU_TRY(run_toeplitz(p, p->ncoil, (const float2*)x_in, p->d_imgwork, (float2*)x_out, p->d_coils, true, st, &summed));
    return summed ? NUFFT_OK : coil_reduce(p, (float2*)x_out, st);
}

static int apply_aha(nufft_plan_t p, bool coils, const float2* in, float2* out, cudaStream_t st) {
    if (p->toep_on) {
        if (coils) return nufft_selfadjoint_toeplitz_coils(p, (const nufft_c64*)in, (nufft_c64*)out, st);
        return nufft_selfadjoint_toeplitz(p, 1, (const nufft_c64*)in, (nufft_c64*)out, st);
    }
    if (coils) return nufft_selfadjoint_coils(p, (const nufft_c64*)in, (nufft_c64*)out, st);
    return nufft_selfadjoint(p, 1, (const nufft_c64*)in, (nufft_c64*)out, st);
}

// operator of the L1TV inner problem, eq. (15): out = mu A^H A z + lam sum_a grad_a^T grad_a z   (mu = 1, lam = 0: A^H A)
struct NormalOp {
    bool coils;
    bool tv;
    float mu, lam;
    bool kspace = false;      // the operator is V^H V on the oversampled grid (the paper's k-space CG, eq. 11)
};
static int apply_op(nufft_plan_t p, const NormalOp& op, const float2* in, float2* out, cudaStream_t st) {
    if (op.kspace) {          // out = V^H (V in), planar grid vectors of prod(K) cells
        NU_TRY(run_interp(p, 1, in, p->d_ywork, st));
        return run_gridding(p, 1, p->d_ywork, out, st);
    }
    NU_TRY(apply_aha(p, op.coils, in, out, st));
    if (op.tv) {
        tv_normal_kernel<<<ew_blocks(p->nimg), 256, 0, st>>>(out, in, op.mu, op.lam, p->N[0], p->N[1]);
        CU_TRY(cudaGetLastError());
        p->launches++;
    }
    return NUFFT_OK;
}

// niter CG steps on op(x) = rhs from the x already in `x` (warm = true) or from 0 (warm = false, x is overwritten).
// r, pv, Ap: work vectors.  hist: device double[niter + 1] or nullptr.
static int cg_run(nufft_plan_t p, const NormalOp& op, const float2* rhs, float2* x, bool warm, int niter, float2* r,
                  float2* pv, float2* Ap, double* hist, cudaStream_t st) {
    const int64_t n = op.kspace ? p->cells : p->nimg;
    const int nb = ew_blocks(n);
    scalars_clear_kernel<<<1, 1, 0, st>>>(p->d_scal);
    if (warm) {
        NU_TRY(apply_op(p, op, x, Ap, st));
        cg_init_kernel<<<nb, 256, 0, st>>>(rhs, Ap, r, pv, n, p->d_scal);
    } else {
        CU_TRY(cudaMemsetAsync(x, 0, (size_t)n * sizeof(float2), st));
        cg_init_kernel<<<nb, 256, 0, st>>>(rhs, nullptr, r, pv, n, p->d_scal);
    }
    cg_shift_kernel<<<1, 1, 0, st>>>(p->d_scal, hist, 1);
    p->launches += 3;
    // One iteration has fixed pointers and scalars that live on the device, so it is one replayable CUDA graph
    // (opts.use_graphs): the first iteration runs eagerly (lazy allocations happen there), the second is captured, the
    // rest are replays.  Per-kernel event profiling needs eager launches.
    auto iteration = [&]() -> int {
        NU_TRY(apply_op(p, op, pv, Ap, st));
        dot_real_kernel<<<nb, 256, 0, st>>>(pv, Ap, n, &p->d_scal->pAp);
        cg_update_xr_kernel<<<nb, 256, 0, st>>>(x, r, pv, Ap, n, p->d_scal);
        cg_update_p_kernel<<<nb, 256, 0, st>>>(pv, r, n, p->d_scal);
        cg_shift_kernel<<<1, 1, 0, st>>>(p->d_scal, hist, 0);
        p->launches += 4;
        return NUFFT_OK;
    };
    const bool graphs = p->opts.use_graphs && !p->prof_on && niter >= 3 && st != nullptr;   // the legacy stream cannot capture
    int k = 0;
    if (niter > 0) {
        const int64_t l0 = p->launches;
        NU_TRY(iteration());
        p->cg_iter_launches = (int)(p->launches - l0);
        k = 1;
    }
    if (graphs) {
        CgGraphKey key;
        std::memset(&key, 0, sizeof(key));
        key.coils = op.coils; key.tv = op.tv; key.mu = op.mu; key.lam = op.lam; key.toep = p->toep_on || op.kspace;
        key.x = x; key.r = r; key.pv = pv; key.Ap = Ap; key.hist = hist; key.stream = (void*)st;
        if (!p->cg_graph || std::memcmp(&key, &p->cg_key, sizeof(key)) != 0) {
            if (p->cg_graph) { cudaGraphExecDestroy(p->cg_graph); p->cg_graph = nullptr; }
            const int64_t l0 = p->launches;
            CU_TRY(cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal));
            const int rc = iteration();
            cudaGraph_t g = nullptr;
            const cudaError_t e = cudaStreamEndCapture(st, &g);
            p->launches = l0;                       // the captured launches did not run
            if (rc != NUFFT_OK || e != cudaSuccess || !g) {
                if (g) cudaGraphDestroy(g);
                (void)cudaGetLastError();
                if (rc != NUFFT_OK) return rc;
                g_last_cuda_error = (int)e;
                return NUFFT_ECUDA;
            }
            const cudaError_t ei = cudaGraphInstantiate(&p->cg_graph, g, 0);
            cudaGraphDestroy(g);
            if (ei != cudaSuccess) { p->cg_graph = nullptr; g_last_cuda_error = (int)ei; (void)cudaGetLastError(); return NUFFT_ECUDA; }
            p->cg_key = key;
        }
        for (; k < niter; ++k) {
            CU_TRY(cudaGraphLaunch(p->cg_graph, st));
            p->launches += p->cg_iter_launches;
        }
    } else {
        for (; k < niter; ++k) NU_TRY(iteration());
    }
    CU_TRY(cudaGetLastError());
    return NUFFT_OK;
}

static int adjoint_any(nufft_plan_t p, bool coils, const float2* y, float2* x, cudaStream_t st) {
    if (coils) return nufft_adjoint_coils(p, (const nufft_c64*)y, (nufft_c64*)x, st);
    return nufft_adjoint(p, 1, (const nufft_c64*)y, (nufft_c64*)x, st);
}

extern "C" int nufft_solve_cg(nufft_plan_t p, int use_coils, const nufft_c64* y, nufft_c64* x, int niter,
                              double* resnorm_host, void* stream) {
    if (!p || wrong_device(p) || !y || !x || niter < 0) return NUFFT_EINVAL;
    const bool coils = use_coils != 0;
    if (coils && p->ncoil < 1) return NUFFT_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    NU_TRY(ensure_solver(p, 4, niter + 1));
    float2* rhs = p->d_solver;
    float2* r = rhs + p->nimg;
    float2* pv = r + p->nimg;
    float2* Ap = pv + p->nimg;
    NU_TRY(adjoint_any(p, coils, (const float2*)y, rhs, st));
    NormalOp op{coils, false, 1.f, 0.f};
    NU_TRY(cg_run(p, op, rhs, (float2*)x, false, niter, r, pv, Ap, p->d_hist, st));
    if (resnorm_host) {
        CU_TRY(cudaMemcpyAsync(resnorm_host, p->d_hist, (size_t)(niter + 1) * sizeof(double), cudaMemcpyDeviceToHost, st));
        CU_TRY(cudaStreamSynchronize(st));
    }
    return NUFFT_OK;
}

// The paper's own CG (eqs. 8-11; reading R24): conjugate gradient on V^H V k = V^H y over the
// oversampled grid, k_0 = 0, exactly niter iterations; then x = S^-1 F^-1 k (normalised inverse FFT, crop, divide by the
// scaling factor).
extern "C" int nufft_solve_cg_kspace(nufft_plan_t p, const nufft_c64* y, nufft_c64* x, int niter, double* resnorm_host,
                                     void* stream) {
    if (!p || wrong_device(p) || !x || (!y && p->M > 0) || niter < 0) return NUFFT_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t n = p->cells;
    if (!p->d_kspace) NU_TRY(dev_alloc((void**)&p->d_kspace, (size_t)5 * n * sizeof(float2), &p->bytes_work));
    if (!p->d_sinv[0]) {
        for (int a = 0; a < p->d; ++a) {
            std::vector<float> s = host::scaling_vector(p->N[a], p->K[a], (double)p->J);
            // 1 / (s K): computed in float64 from the float64 scaling factor, rounded once
            const double beta = host::kb_beta((double)p->J, (double)p->K[a] / (double)p->N[a]);
            for (int i = 0; i < p->N[a]; ++i)
                s[i] = (float)(host::kb_Phi(((double)i - 0.5 * p->N[a]) / (double)p->K[a], (double)p->J, beta) / (double)p->K[a]);
            NU_TRY(dev_upload(&p->d_sinv[a], s, &p->bytes_plan));
        }
    }
    NU_TRY(ensure_solver(p, 0, niter + 1));
    float2 *rhs = p->d_kspace, *k = rhs + n, *r = k + n, *pv = r + n, *Ap = pv + n;
    NU_TRY(run_gridding(p, 1, (const float2*)y, rhs, st));                 // V^H y
    NormalOp op{false, false, 1.f, 0.f, true};
    NU_TRY(cg_run(p, op, rhs, k, false, niter, r, pv, Ap, p->d_hist, st));
    p->inv_scale = true;                                                     // x = S^-1 F^-1 k  (eq. 10); k is consumed
    const int rc = run_fft_scale(p, 1, k, (float2*)x, nullptr, st);
    p->inv_scale = false;
    NU_TRY(rc);
    if (resnorm_host) {
        CU_TRY(cudaMemcpyAsync(resnorm_host, p->d_hist, (size_t)(niter + 1) * sizeof(double), cudaMemcpyDeviceToHost, st));
        CU_TRY(cudaStreamSynchronize(st));
    }
    return NUFFT_OK;
}

extern "C" int nufft_solve_l1tv_ols(nufft_plan_t p, int use_coils, const nufft_c64* y, nufft_c64* x, double mu,
                                    double lam, int n_outer, int n_inner, int n_cg, void* stream) {
    if (!p || wrong_device(p) || !y || !x || n_outer < 0 || n_inner < 0 || n_cg < 0 || p->d != 2 || lam < 0.0) return NUFFT_EINVAL;
    const bool coils = use_coils != 0;
    if (coils && p->ncoil < 1) return NUFFT_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t n = p->nimg;
    NU_TRY(ensure_solver(p, 12, 1));
    float2* v = p->d_solver;
    float2 *ahy_s = v, *ahy_k = v + n, *rhs = v + 2 * n, *r = v + 3 * n, *pv = v + 4 * n, *Ap = v + 5 * n;
    float2 *d0 = v + 6 * n, *b0 = v + 7 * n, *d1 = v + 8 * n, *b1 = v + 9 * n, *xs = v + 10 * n, *tmp = v + 11 * n;
    const int nb = ew_blocks(n);
    // A^H y and the problem scale c = 1 / max |A^H y|   (R17)
    NU_TRY(adjoint_any(p, coils, (const float2*)y, tmp, st));
    scalars_clear_kernel<<<1, 1, 0, st>>>(p->d_scal);
    maxabs_kernel<<<nb, 256, 0, st>>>(tmp, n, p->d_scal);
    p->launches += 2;
    double mx = 0.0;
    CU_TRY(cudaMemcpyAsync(&mx, &p->d_scal->maxabs, sizeof(double), cudaMemcpyDeviceToHost, st));
    CU_TRY(cudaStreamSynchronize(st));
    if (!(mx > 0.0)) {   // A^H y = 0: the solution is 0
        CU_TRY(cudaMemsetAsync(x, 0, (size_t)n * sizeof(float2), st));
        return NUFFT_OK;
    }
    const float c = (float)(1.0 / mx);
    scale_kernel<<<nb, 256, 0, st>>>(ahy_s, tmp, c, n);
    CU_TRY(cudaMemcpyAsync(ahy_k, ahy_s, (size_t)n * sizeof(float2), cudaMemcpyDeviceToDevice, st));
    CU_TRY(cudaMemsetAsync(d0, 0, (size_t)4 * n * sizeof(float2), st));     // d0, b0, d1, b1 are contiguous
    CU_TRY(cudaMemsetAsync(xs, 0, (size_t)n * sizeof(float2), st));
    p->launches += 1;
    const float fmu = (float)mu, flam = (float)lam;
    const float thr = (lam > 0.0) ? (float)(1.0 / lam) : -1.0f;
    NormalOp op{coils, true, fmu, flam};
    for (int o = 0; o < n_outer; ++o) {
        for (int i = 0; i < n_inner; ++i) {
            tv_rhs_kernel<<<nb, 256, 0, st>>>(rhs, ahy_k, d0, b0, d1, b1, fmu, flam, p->N[0], p->N[1]);   // eq. (16)
            p->launches++;
            NU_TRY(cg_run(p, op, rhs, xs, true, n_cg, r, pv, Ap, nullptr, st));                           // eq. (17)
            tv_shrink_kernel<<<nb, 256, 0, st>>>(xs, d0, b0, d1, b1, thr, p->N[0], p->N[1]);             // eqs. (18)-(21)
            p->launches++;
        }
        NU_TRY(apply_aha(p, coils, xs, tmp, st));
        tv_outer_kernel<<<nb, 256, 0, st>>>(ahy_k, ahy_s, tmp, n);                                        // eq. (22)
        p->launches++;
    }
    scale_kernel<<<nb, 256, 0, st>>>((float2*)x, xs, (float)mx, n);
    p->launches++;
    CU_TRY(cudaGetLastError());
    return NUFFT_OK;
}

extern "C" int nufft_solve_l1tv_lad(nufft_plan_t p, int use_coils, const nufft_c64* y, nufft_c64* x, double mu,
                                    double lam, int n_outer, int n_inner, int n_cg, void* stream) {
    if (!p || wrong_device(p) || !y || !x || n_outer < 0 || n_inner < 0 || n_cg < 0 || p->d != 2 || lam < 0.0 || mu < 0.0) return NUFFT_EINVAL;
    const bool coils = use_coils != 0;
    if (coils && p->ncoil < 1) return NUFFT_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t n = p->nimg;
    NU_TRY(ensure_solver(p, 15, 1));
    float2* v = p->d_solver;
    float2 *ahy_s = v, *ahy_k = v + n, *rhs = v + 2 * n, *r = v + 3 * n, *pv = v + 4 * n, *Ap = v + 5 * n;
    float2 *d0 = v + 6 * n, *b0 = v + 7 * n, *d1 = v + 8 * n, *b1 = v + 9 * n, *df = v + 10 * n, *bf = v + 11 * n;
    float2 *xs = v + 12 * n, *tmp = v + 13 * n, *prep = v + 14 * n;
    const int nb = ew_blocks(n);
    NU_TRY(adjoint_any(p, coils, (const float2*)y, tmp, st));
    scalars_clear_kernel<<<1, 1, 0, st>>>(p->d_scal);
    maxabs_kernel<<<nb, 256, 0, st>>>(tmp, n, p->d_scal);
    p->launches += 2;
    double mx = 0.0;
    CU_TRY(cudaMemcpyAsync(&mx, &p->d_scal->maxabs, sizeof(double), cudaMemcpyDeviceToHost, st));
    CU_TRY(cudaStreamSynchronize(st));
    if (!(mx > 0.0)) {
        CU_TRY(cudaMemsetAsync(x, 0, (size_t)n * sizeof(float2), st));
        return NUFFT_OK;
    }
    scale_kernel<<<nb, 256, 0, st>>>(ahy_s, tmp, (float)(1.0 / mx), n);
    CU_TRY(cudaMemcpyAsync(ahy_k, ahy_s, (size_t)n * sizeof(float2), cudaMemcpyDeviceToDevice, st));
    CU_TRY(cudaMemsetAsync(d0, 0, (size_t)7 * n * sizeof(float2), st));     // d0, b0, d1, b1, df, bf, xs are contiguous
    p->launches += 1;
    const float fmu = (float)mu, flam = (float)lam;
    const float thr = (lam > 0.0) ? (float)(1.0 / lam) : -1.0f;
    const float thr_f = (mu > 0.0) ? (float)(1.0 / mu) : -1.0f;
    NormalOp op{coils, true, fmu, flam};
    for (int o = 0; o < n_outer; ++o) {
        for (int i = 0; i < n_inner; ++i) {
            lad_prep_kernel<<<nb, 256, 0, st>>>(prep, ahy_k, df, bf, n);                                   // eq. (25)
            tv_rhs_kernel<<<nb, 256, 0, st>>>(rhs, prep, d0, b0, d1, b1, fmu, flam, p->N[0], p->N[1]);
            NU_TRY(cg_run(p, op, rhs, xs, true, n_cg, r, pv, Ap, nullptr, st));                            // eq. (26)
            tv_shrink_kernel<<<nb, 256, 0, st>>>(xs, d0, b0, d1, b1, thr, p->N[0], p->N[1]);               // (27)-(28), (30)-(31)
            NU_TRY(apply_aha(p, coils, xs, tmp, st));
            lad_data_kernel<<<nb, 256, 0, st>>>(tmp, ahy_s, df, bf, thr_f, n);                             // (29), (32)
            p->launches += 4;
        }
        if (n_inner == 0) NU_TRY(apply_aha(p, coils, xs, tmp, st));
        tv_outer_kernel<<<nb, 256, 0, st>>>(ahy_k, ahy_s, tmp, n);                                         // eq. (33)
        p->launches++;
    }
    scale_kernel<<<nb, 256, 0, st>>>((float2*)x, xs, (float)mx, n);
    p->launches++;
    CU_TRY(cudaGetLastError());
    return NUFFT_OK;
}

// ------------------------------------------------------------------------------------------------------------
extern "C" const char* nufft_strerror(int code) {
    switch (code) {
        case NUFFT_OK: return "ok";
        case NUFFT_EINVAL: return "invalid argument or unsupported configuration";
        case NUFFT_ENOMEM: return "out of memory";
        case NUFFT_ECUDA: return "CUDA runtime error (see nufft_last_cuda_error)";
        case NUFFT_ERANGE: return "non-finite sample location";
        case NUFFT_ESTATE: return "missing state (coil maps not set)";
        case NUFFT_ETOOBIG: return "oversampled grid larger than the static scratch of nufft_adjoint_noalloc (NUFFT_NOALLOC_MAX_CELLS cells)";
    }
    return "unknown error";
}
extern "C" int nufft_last_cuda_error(void) { return g_last_cuda_error; }
extern "C" const char* nufft_version(void) { return "nufft-b200 0.1 (sm_100a)"; }
