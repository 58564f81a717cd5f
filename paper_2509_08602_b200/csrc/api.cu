// C ABI of libadmm_b200.so (include/admm_b200.h): setup (S0-S2), the batched solve loop (H1-H6 of DESIGN.md)
// with per-plan convergence masking + compaction, and the parity / timing hooks.  Host orchestration only:
// every step of the path runs in the kernels of gemm_tc.cu / kernels.cu (+ cuBLAS/cuSOLVER fp64 for the one-off
// factorisation of S).
#include <cublas_v2.h>
#include <cusolverDn.h>

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <type_traits>

#include "admm_internal.h"

void launch_simt_k1(admm_handle* h, int slot0, int nact, int n_mma, int splits, cudaStream_t s);

namespace {

std::string g_setup_err = "no error";

inline int64_t cdiv(int64_t a, int64_t b) { return (a + b - 1) / b; }
inline int64_t round_up(int64_t a, int64_t b) { return cdiv(a, b) * b; }
double now_ms() {
    return std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now().time_since_epoch()).count();
}

#define CU_TRY(h, expr)                                                                       \
    do {                                                                                      \
        cudaError_t _e = (expr);                                                              \
        if (_e != cudaSuccess) {                                                              \
            (h)->err = std::string(#expr) + ": " + cudaGetErrorString(_e);                   \
            return (_e == cudaErrorMemoryAllocation) ? ADMM_ENOMEM : ADMM_ECUDA;              \
        }                                                                                     \
    } while (0)

template <typename T>
admm_status dev_alloc(admm_handle* h, T** p, int64_t count) {
    if (*p) { cudaFree(*p); *p = nullptr; }
    cudaError_t e = cudaMalloc(reinterpret_cast<void**>(p), (size_t)std::max<int64_t>(count, 1) * sizeof(T));
    if (e != cudaSuccess) {
        char buf[128];
        snprintf(buf, sizeof buf, "cudaMalloc of %lld bytes failed: %s", (long long)(count * (int64_t)sizeof(T)), cudaGetErrorString(e));
        h->err = buf;
        *p = nullptr;
        return ADMM_ENOMEM;
    }
    return ADMM_OK;
}
#define ST_TRY(expr) do { admm_status _s = (expr); if (_s != ADMM_OK) return _s; } while (0)

bool is_device_ptr(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

// ---- unit tables ------------------------------------------------------------------------------------------
// K3: the 128-row tiles of Phi (aligned: the big operand is stored tile-major) are dealt evenly to the CTAs.
void build_units_k3(int64_t N, int64_t n, int sm, int kblk, std::vector<TcUnit>& units, std::vector<int32_t>& begin) {
    const int64_t tiles = cdiv(N, kTileM);
    const int grid = (int)std::min<int64_t>(sm, tiles);
    const int kb = (int)cdiv(n, kblk);
    units.clear(); begin.assign(1, 0);
    for (int c = 0; c < grid; ++c) {
        for (int64_t t = tiles * c / grid; t < tiles * (c + 1) / grid; ++t) {
            const int64_t row0 = t * kTileM;
            units.push_back(TcUnit{(int32_t)row0, (int32_t)std::min<int64_t>(kTileM, N - row0), 0, kb, 0, 0});
        }
        begin.push_back((int32_t)units.size());
    }
}
// K1: slab-major stream-K.  Work = (m-tile of 128 time variables) x (k-blocks of 32 points).  The k-range is cut into
// slabs whose slice of the small operand G (hi + lo, all plans of a pass) fits comfortably in L2; inside a slab the work is
// linearised m-tile-major and cut into `grid` equal contiguous pieces (a piece that crosses an m-tile boundary becomes two
// units).  All CTAs are inside the same slab at the same time, so G is read from HBM once per iteration instead of once
// per m-tile (measured at config 2 before this ordering: K1 took 7.6 ms against K3's 4.8 ms for the same Phi bytes).
// Every unit writes its own partial-sum slot; the slots of one m-tile are numbered contiguously (mtile_slot_begin).
void build_units_k1(int64_t N, int64_t n, int sm, int kblk, int n_mma_max, int slab_kb, std::vector<TcUnit>& units,
                    std::vector<int32_t>& begin, std::vector<int32_t>& mtile_slot_begin) {
    const int64_t T = cdiv(n, kTileM);
    const int64_t KB = cdiv(N, kblk);
    const int grid = (int)std::min<int64_t>(sm, T * std::max<int64_t>(1, KB / 8));
    const int64_t g_bytes_per_kb = (int64_t)2 * n_mma_max * 128;      // hi + lo rows of 128 bytes
    int64_t slabs = 1;
    if (slab_kb > 0) slabs = cdiv(KB, slab_kb);
    else if (KB * g_bytes_per_kb > (64ll << 20)) slabs = cdiv(KB * g_bytes_per_kb, 32ll << 20);
    units.clear(); begin.assign(1, 0);
    std::vector<std::vector<TcUnit>> per_cta(grid);
    for (int64_t sl = 0; sl < slabs; ++sl) {
        const int64_t kb_lo = KB * sl / slabs, kb_hi = KB * (sl + 1) / slabs, len = kb_hi - kb_lo;
        if (len <= 0) continue;
        const int64_t W = T * len;
        for (int c = 0; c < grid; ++c) {
            int64_t lo = W * c / grid; const int64_t hi = W * (c + 1) / grid;
            while (lo < hi) {
                const int64_t mt = lo / len, off = lo % len;
                const int64_t take = std::min(hi - lo, len - off);
                const int rows = (int)std::min<int64_t>(kTileM, n - mt * kTileM);
                per_cta[c].push_back(TcUnit{(int32_t)(mt * kTileM), rows, (int32_t)(kb_lo + off), (int32_t)take, 0, 0});
                lo += take;
            }
        }
    }
    // slot ids: m-tile-major
    std::vector<int32_t> count(T, 0);
    for (auto& v : per_cta) for (auto& u : v) count[u.row0 / kTileM]++;
    mtile_slot_begin.assign(T + 1, 0);
    for (int64_t mt = 0; mt < T; ++mt) mtile_slot_begin[mt + 1] = mtile_slot_begin[mt] + count[mt];
    std::vector<int32_t> next(mtile_slot_begin.begin(), mtile_slot_begin.end() - 1);
    for (auto& v : per_cta) {
        for (auto& u : v) { u.slot = next[u.row0 / kTileM]++; units.push_back(u); }
        begin.push_back((int32_t)units.size());
    }
}

struct EvPair { cudaEvent_t a, b; int kind; };

struct Profiler {
    bool on = false;
    std::vector<EvPair> live;
    std::vector<EvPair> pool;
    void begin(admm_handle* h, int kind) {
        if (!on) return;
        EvPair e;
        if (!pool.empty()) { e = pool.back(); pool.pop_back(); } else { cudaEventCreate(&e.a); cudaEventCreate(&e.b); }
        e.kind = kind;
        cudaEventRecord(e.a, h->stream);
        live.push_back(e);
    }
    void end(admm_handle* h) {
        if (!on) return;
        cudaEventRecord(live.back().b, h->stream);
    }
    void harvest(admm_handle* h) {          // stream must be synchronised
        for (auto& e : live) {
            float ms = 0; cudaEventElapsedTime(&ms, e.a, e.b);
            h->ktimes.total_ms[e.kind] += ms; h->ktimes.launches[e.kind]++;
            pool.push_back(e);
        }
        live.clear();
    }
    ~Profiler() { for (auto& e : pool) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); } }
};

void free_all(admm_handle* h) {
    void* ptrs[] = {h->d_phi, h->d_phiT, h->d_phi_t, h->d_phiT_t, h->d_csr_ptr, h->d_csrT_ptr, h->d_csr_col, h->d_csrT_col, h->d_csr_val, h->d_csrT_val, h->d_small_t, h->d_point_class, h->d_R, h->d_Rb, h->d_bot, h->d_Sinv, h->d_s1, h->d_ghi, h->d_s2, h->d_rhs,
                    h->d_vhi, h->d_partial, h->d_resid1, h->d_resid2, h->d_hinge, h->d_mask, h->d_slot_plan,
                    h->d_utab, h->d_crtab, h->d_beta, h->d_rho, h->d_active_counts, h->d_conv_flags, h->d_bact, h->d_moves,
                    h->d_nmoves, h->d_iters_plan, h->d_res_plan, h->d_wnorm, h->d_t_f32, h->d_obj, h->d_plan_slot, h->d_tout,
                    h->d_qbuf, h->d_units_k1, h->d_cta_begin_k1, h->d_mtile_slot_begin, h->d_units_k3, h->d_cta_begin_k3};
    for (void* p : ptrs) if (p) cudaFree(p);
    if (h->h_bact_ring) cudaFreeHost(h->h_bact_ring);
    for (cudaEvent_t e : h->bact_ev) if (e) cudaEventDestroy(e);
}

EpiParams base_epi(admm_handle* h) {
    EpiParams ep{};
    ep.N = h->N; ep.n = h->n; ep.ldN = h->ldN; ep.ldn = h->ldn;
    ep.partial = h->d_partial;
    ep.point_class = h->d_point_class;
    ep.mask = h->has_mask ? h->d_mask : nullptr;
    ep.slot_plan = h->d_slot_plan;
    ep.mask_words = h->mask_words;
    ep.utab = h->d_utab; ep.crtab = h->d_crtab;
    for (int k = 0; k < kMaxClasses; ++k) { ep.a_cls[k] = 0; ep.sense[k] = 0; ep.thr[k] = 0; }
    for (int k = 0; k < h->n_classes; ++k) {
        ep.a_cls[k] = (float)((double)h->classes[k].sense / ((double)h->classes[k].threshold * (double)h->class_count[k]));
        ep.sense[k] = (float)h->classes[k].sense;
        ep.thr[k] = h->classes[k].threshold;
    }
    ep.s1 = h->d_s1; ep.g_hi = h->d_ghi; ep.g_lo = h->d_glo;
    ep.resid_partial = nullptr; ep.hinge_partial = h->d_hinge;
    ep.small_bf16 = h->opt.storage == ADMM_STORAGE_BF16 ? 1 : 0;
    ep.bact_dev = nullptr;          // set by the iteration loop only: start-up, finalise and the probes act on exact slot ranges
    return ep;
}

int mma_passes(const admm_handle* h) { return h->opt.storage == ADMM_STORAGE_FP32_3XTF32 ? 3 : 2; }
// fp32 path: drain the hi.hi TMEM accumulator every k-block (32 elements of K, 4 MMAs) -- see gemm_tc.cu
int chunk_kb(const admm_handle* h) {
    if (h->opt.kernel_path != ADMM_PATH_TCGEN05) return 0;
    if (h->opt.drain_kb < 0) return 0;
    if (h->opt.drain_kb > 0) return h->opt.drain_kb;
    // every k-block (4 accumulations), with the mean truncation loss put back (TcLaunch::debias): K = 50 iterates at config 1 sit
    // at 4e-5 / 5e-5 of the oracle's.  Longer chunks are faster (2: K1 / K3 101 / 134 -> 93 / 123 us) but their rounding noise grows
    // with the chunk (t of the degenerate plan of config 0: 8.7e-5 -> 1.3e-4), and with two MMA issuers a chunk of several k-blocks
    // would be accumulated by both in an order that is not fixed (gemm_tc.cu falls back to one issuer then).  bf16 storage has a
    // 1e-2 budget and drains every 4.
    return h->opt.storage == ADMM_STORAGE_BF16 ? 4 : 1;
}
// plans per contraction pass
int max_pass(const admm_handle* h) {
    return (mma_passes(h) == 3 && h->opt.kernel_path == ADMM_PATH_TCGEN05) ? 96 : kMaxMmaN;
}

// one contraction pass over slots [slot0, slot0 + nact): big operand + small hi/lo rows starting at slot0.
// The four tensor maps of a (contraction, slot0, n_mma) are encoded once per batch allocation and kept (an encode costs a few
// microseconds of host time, eight of them per iteration were a visible share of a 0.2 ms iteration).
admm_status contract(admm_handle* h, int epi, int slot0, int nact, const float* small_hi, const float* small_lo,
                     bool resid, float* qraw = nullptr, bool live_from_device = false) {
    const int n_mma = (int)round_up(nact, 16);
    TcLaunch L{};
    const bool k1 = (epi == EPI_K1_PARTIAL);
    const int64_t big_rows = k1 ? h->n : h->N, big_cols = k1 ? h->N : h->n, big_ld = k1 ? h->ldN : h->ldn;
    // big operand: tile-major [row tiles][k-blocks][128 rows][128 bytes] seen as a 2-D tensor of 128-byte rows
    const bool bf16 = h->opt.storage == ADMM_STORAGE_BF16;
    const int eb = bf16 ? 2 : 4, kblk = h->kblk;
    const int64_t kb_total = cdiv(big_cols, kblk), tiled_rows = cdiv(big_rows, kTileM) * kb_total * kTileM;
    const int kind = k1 ? 0 : 1;          // the small operand of K3 / objective / probe(1) is always the V buffer pair
    const admm_handle::MapKey* hit = nullptr;
    for (const auto& m : h->map_cache) if (m.kind == kind && m.slot0 == slot0 && m.n_mma == n_mma) { hit = &m; break; }
    if (!hit) {
        admm_handle::MapKey m{}; m.kind = kind; m.slot0 = slot0; m.n_mma = n_mma;
        ST_TRY(tc_make_map(h, &m.big, k1 ? h->d_phiT_t : h->d_phi_t, tiled_rows, kblk, kblk, kBoxRows, eb));
        ST_TRY(tc_make_map(h, &m.big128, k1 ? h->d_phiT_t : h->d_phi_t, tiled_rows, kblk, kblk, kTileM, eb));
        // the small operand has Bpad rows allocated (row pitch big_ld * 4 bytes whatever the element type); rows >= nact of the
        // box are dead columns of D
        ST_TRY(tc_make_map(h, &m.hi, small_hi + (int64_t)slot0 * big_ld, h->Bpad - slot0, big_cols, bf16 ? 2 * big_ld : big_ld, n_mma, eb));
        ST_TRY(tc_make_map(h, &m.lo, small_lo + (int64_t)slot0 * big_ld, h->Bpad - slot0, big_cols, bf16 ? 2 * big_ld : big_ld, n_mma, eb));
        h->map_cache.push_back(m);
        hit = &h->map_cache.back();
    }
    L.map_big = hit->big; L.map_big128 = hit->big128; L.map_small_hi = hit->hi; L.map_small_lo = hit->lo;
    L.big_kb_total = (int32_t)kb_total;
    L.kblk = kblk; L.mma_kind = bf16 ? 1 : 0;
    L.units = k1 ? h->d_units_k1 : h->d_units_k3;
    L.cta_unit_begin = k1 ? h->d_cta_begin_k1 : h->d_cta_begin_k3;
    L.grid = k1 ? h->grid_k1 : h->grid_k3;
    L.mma_passes = mma_passes(h);
    L.epi = epi;
    L.chunk_kb = chunk_kb(h);
    // measured on B200 (tests/test_gpu_parity.py test_accumulation_is_unbiased): a chunk of m tcgen05.mma accumulations from a
    // cleared accumulator comes out low by ~3.5e-8 m of its value (4 MMAs per k-block => 1.4e-7 at drain_kb = 1).  Off by default:
    // at drain_kb = 1 the loss is a common scale factor of 1 - 1.4e-7 on both products, far below the LP's accuracy, and putting
    // it back moved the K = 50 iterates by less than their rounding noise (z 6.8e-5 -> 4.2e-5, t of the degenerate plan
    // 4.8e-4 -> 5.3e-4 at config 1); it is what makes longer drain intervals usable (drain_kb = 4: z 2.1e-4 -> 6.5e-5).
    L.debias = (L.chunk_kb > 0 && h->opt.accum_debias > 0) ? 1.4e-7f * (float)L.chunk_kb * (h->opt.accum_debias / 100.f) : 0.f;
    L.ep = base_epi(h);
    L.ep.slot0 = slot0; L.ep.n_slots_active = nact; L.ep.n_mma = n_mma;
    L.ep.bact_dev = live_from_device ? h->d_bact : nullptr;
    L.ep.resid_partial = resid ? h->d_resid1 : nullptr;
    L.ep.qraw = qraw;
    return tc_launch(h, L);
}
admm_status contract_raw(admm_handle* h, int nact, const float* hi, const float* lo, float* qbuf) {
    return contract(h, EPI_RAW, 0, nact, hi, lo, false, qbuf);
}

}  // namespace

// ================================================================================================ C ABI
extern "C" {

void admm_default_options(admm_options* opt) {
    if (!opt) return;
    memset(opt, 0, sizeof(*opt));
    opt->storage = ADMM_STORAGE_FP32_3XTF32;
    opt->kernel_path = ADMM_PATH_TCGEN05;
    opt->check_every = 10;
    opt->eps_abs = 1e-6f;
    opt->compaction = 1;
    opt->presolve = 1;
}

const char* admm_version(void) { return "paper_2509_08602_b200 0.1 sm_100a"; }

const char* admm_last_error(const admm_handle* h) { return h ? h->err.c_str() : g_setup_err.c_str(); }

int64_t admm_last_launch_count(const admm_handle* h) { return h ? h->launch_count : 0; }

void admm_destroy(admm_handle* h) {
    if (!h) return;
    cudaSetDevice(h->opt.device);
    free_all(h);
    delete h;
}

static admm_status setup_impl(admm_handle* h, const float* phi, int32_t phi_on_device, int64_t N, int64_t n, int64_t ld,
                              const uint8_t* point_class, const admm_class* classes, int32_t n_classes) {
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0) { cudaGetLastError(); h->err = "no CUDA device (this library has no CPU fallback)"; return ADMM_ECUDA; }
    if (h->opt.device < 0 || h->opt.device >= ndev) { h->err = "opt.device out of range"; return ADMM_EINVAL; }
    CU_TRY(h, cudaSetDevice(h->opt.device));
    cudaDeviceProp prop;
    CU_TRY(h, cudaGetDeviceProperties(&prop, h->opt.device));
    if (prop.major != 10) { h->err = "device is not sm_100 (Blackwell B200): tcgen05/TMEM kernels cannot run"; return ADMM_ECUDA; }
    h->sm_count = prop.multiProcessorCount;
    h->stream = reinterpret_cast<cudaStream_t>(h->opt.stream);
    cudaStream_t st = h->stream;

    h->N = N; h->n = n; h->ldn = round_up(n, 4); h->ldN = round_up(N, 4);
    h->n_classes = n_classes;
    for (int k = 0; k < n_classes; ++k) { h->classes[k] = classes[k]; h->class_count[k] = 0; }
    h->h_point_class.assign(point_class, point_class + N);
    for (int64_t i = 0; i < N; ++i) {
        if (point_class[i] >= n_classes) { h->err = "point_class entry >= n_classes"; return ADMM_EINVAL; }
        h->class_count[point_class[i]]++;
    }
    for (int k = 0; k < n_classes; ++k)
        if (h->class_count[k] == 0) { h->err = "a class has no points"; return ADMM_EINVAL; }

    const double t0 = now_ms();
    // ---- S0: Phi row-major [N][ldn] (setup), then the resident tile-major copies of Phi and Phi^T
    const bool tc_path = h->opt.kernel_path == ADMM_PATH_TCGEN05;
    const bool bf16 = h->opt.storage == ADMM_STORAGE_BF16;
    h->kblk = bf16 ? 64 : kBlockK;
    const int64_t rtN = cdiv(N, kTileM), rtn = cdiv(n, kTileM), kbN = cdiv(N, h->kblk), kbn = cdiv(n, h->kblk);
    if (std::max(rtN * kbn, rtn * kbN) * kTileM >= (1ll << 31)) { h->err = "Phi too large for 32-bit tile coordinates"; return ADMM_EINVAL; }
    if (std::max(rtN, rtn) > 65535) { h->err = "more than 65535 row tiles of 128: N, n must be below 8388480"; return ADMM_EINVAL; }   // gridDim.y of the packing kernels
    ST_TRY(dev_alloc(h, &h->d_phi, N * h->ldn));
    ST_TRY(dev_alloc(h, &h->d_point_class, N));
    CU_TRY(h, cudaMemsetAsync(h->d_phi, 0, (size_t)N * h->ldn * 4, st));
    CU_TRY(h, cudaMemcpy2DAsync(h->d_phi, (size_t)h->ldn * 4, phi, (size_t)ld * 4, (size_t)n * 4, (size_t)N,
                                phi_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st));
    CU_TRY(h, cudaMemcpyAsync(h->d_point_class, point_class, (size_t)N, cudaMemcpyHostToDevice, st));
    if (h->opt.storage == ADMM_STORAGE_CSR) ST_TRY(csr_threshold(h));
    // reduced storage: Phi is rounded ONCE here, so S below is formed from the matrix the kernels consume (SURVEY H-c)
    if (h->opt.storage == ADMM_STORAGE_FP32_TF32) launch_round_tf32(h->d_phi, N * h->ldn, st);
    if (bf16) launch_round_bf16(h->d_phi, N * h->ldn, st);
    if (tc_path) {
        // every tile is 128 rows x 128 bytes = 16 KB = 4096 floats, whatever the element type
        const bool need_T = !h->opt.dose_only;          // a dose-only handle never forms Phi^T G
        ST_TRY(dev_alloc(h, &h->d_phi_t, rtN * kbn * kTileM * kBlockK));
        if (need_T) ST_TRY(dev_alloc(h, &h->d_phiT_t, rtn * kbN * kTileM * kBlockK));
        if (bf16) {
            launch_pack_tiles_bf16(h->d_phi, N, n, h->ldn, false, h->d_phi_t, st);
            if (need_T) launch_pack_tiles_bf16(h->d_phi, N, n, h->ldn, true, h->d_phiT_t, st);
        } else {
            launch_pack_tiles(h->d_phi, N, n, h->ldn, false, h->d_phi_t, st);
            if (need_T) launch_pack_tiles(h->d_phi, N, n, h->ldn, true, h->d_phiT_t, st);
        }
    } else {
        ST_TRY(dev_alloc(h, &h->d_phiT, n * h->ldN));
        CU_TRY(h, cudaMemsetAsync(h->d_phiT, 0, (size_t)n * h->ldN * 4, st));
        launch_transpose(h->d_phi, N, n, h->ldn, h->d_phiT, h->ldN, st);
    }
    CU_TRY(h, cudaStreamSynchronize(st));
    const double t1 = now_ms();

    if (h->opt.dose_only) {
        // only Phi . T products will run on this handle (admm_dose): no S, no factorisation, only the K3 work decomposition
        if (tc_path) { cudaFree(h->d_phi); h->d_phi = nullptr; }
        if (tc_path) ST_TRY(tc_init(h));
        std::vector<TcUnit> u; std::vector<int32_t> b;
        build_units_k3(N, n, h->sm_count, h->kblk, u, b);
        h->grid_k3 = (int)b.size() - 1;
        ST_TRY(dev_alloc(h, &h->d_units_k3, (int64_t)u.size()));
        ST_TRY(dev_alloc(h, &h->d_cta_begin_k3, (int64_t)b.size()));
        CU_TRY(h, cudaMemcpy(h->d_units_k3, u.data(), u.size() * sizeof(TcUnit), cudaMemcpyHostToDevice));
        CU_TRY(h, cudaMemcpy(h->d_cta_begin_k3, b.data(), b.size() * 4, cudaMemcpyHostToDevice));
        h->grid_k1 = 1; h->slots_k1 = 1;
        h->ms[0] = t1 - t0; h->ms[1] = 0; h->ms[2] = 0; h->ms[3] = now_ms() - t0;
        return ADMM_OK;
    }

    // ---- S1: M = (A D)(A D)^T = Phi^T diag(a^2) Phi in fp64, then R and S = I + R M R
    ST_TRY(dev_alloc(h, &h->d_R, n));
    ST_TRY(dev_alloc(h, &h->d_Sinv, n * n));
    double a_cls_h[kMaxClasses] = {0};
    for (int k = 0; k < n_classes; ++k)
        a_cls_h[k] = (double)classes[k].sense / ((double)classes[k].threshold * (double)h->class_count[k]);
    double* d_acls = nullptr; double* d_chunk = nullptr;
    cublasHandle_t cb = nullptr; cusolverDnHandle_t cs = nullptr;
    // released on EVERY way out of this function (the early returns of ST_TRY / CU_TRY included)
    struct SetupScratch {
        double*& acls; double*& chunk; cublasHandle_t& cb; cusolverDnHandle_t& cs;
        void release() {
            if (cb) { cublasDestroy(cb); cb = nullptr; }
            if (cs) { cusolverDnDestroy(cs); cs = nullptr; }
            if (acls) { cudaFree(acls); acls = nullptr; }
            if (chunk) { cudaFree(chunk); chunk = nullptr; }
        }
        ~SetupScratch() { release(); }
    } scratch{d_acls, d_chunk, cb, cs};
    auto cleanup = [&]() { scratch.release(); };
    ST_TRY(dev_alloc(h, &d_acls, kMaxClasses));
    CU_TRY(h, cudaMemcpyAsync(d_acls, a_cls_h, sizeof a_cls_h, cudaMemcpyHostToDevice, st));
    const int64_t chunk = std::max<int64_t>(256, std::min<int64_t>(N, (int64_t)(512ll << 20) / (n * 8)));
    ST_TRY(dev_alloc(h, &d_chunk, chunk * n));
    if (cublasCreate(&cb) != CUBLAS_STATUS_SUCCESS) { cleanup(); h->err = "cublasCreate failed"; return ADMM_ECUDA; }
    cublasSetStream(cb, st);
    for (int64_t r0 = 0; r0 < N; r0 += chunk) {
        const int64_t rows = std::min(chunk, N - r0);
        launch_scale_rows_to_f64(h->d_phi, h->ldn, r0, rows, n, h->d_point_class, d_acls, d_chunk, st);
        const double one = 1.0, beta = (r0 == 0) ? 0.0 : 1.0;
        // row-major chunk [rows][n] == column-major (n x rows); C (n x n) += Y Y^T, lower triangle (column-major)
        if (cublasDsyrk(cb, CUBLAS_FILL_MODE_LOWER, CUBLAS_OP_N, (int)n, (int)rows, &one, d_chunk, (int)n, &beta,
                        h->d_Sinv, (int)n) != CUBLAS_STATUS_SUCCESS) { cleanup(); h->err = "cublasDsyrk failed"; return ADMM_ECUDA; }
    }
    launch_finish_S(h->d_Sinv, n, h->d_R, st);
    if (cudaStreamSynchronize(st) != cudaSuccess) { cleanup(); h->err = "S formation failed"; return ADMM_ECUDA; }
    if (tc_path) { cudaFree(h->d_phi); h->d_phi = nullptr; }      // only the tile-major copies stay resident
    if (h->opt.storage == ADMM_STORAGE_CSR) {
        ST_TRY(csr_build(h));
        if (cudaStreamSynchronize(st) != cudaSuccess) { cleanup(); h->err = "CSR build failed"; return ADMM_ECUDA; }
        cudaFree(h->d_phi); h->d_phi = nullptr; cudaFree(h->d_phiT); h->d_phiT = nullptr;
        ST_TRY(dev_alloc(h, &h->d_small_t, std::max(N, n) * (int64_t)kMaxMmaN));
        h->ms[7] = (double)h->csr_nnz / ((double)N * (double)n);
    }
    const double t2 = now_ms();

    // ---- S2: Cholesky + explicit inverse in fp64, shared by every plan and every rho (:222)
    if (cusolverDnCreate(&cs) != CUSOLVER_STATUS_SUCCESS) { cleanup(); h->err = "cusolverDnCreate failed"; return ADMM_ECUDA; }
    cusolverDnSetStream(cs, st);
    int lwork1 = 0, lwork2 = 0;
    cusolverDnDpotrf_bufferSize(cs, CUBLAS_FILL_MODE_LOWER, (int)n, h->d_Sinv, (int)n, &lwork1);
    cusolverDnDpotri_bufferSize(cs, CUBLAS_FILL_MODE_LOWER, (int)n, h->d_Sinv, (int)n, &lwork2);
    double* d_work = nullptr; int* d_info = nullptr;
    const int lwork = std::max(lwork1, lwork2);
    if (cudaMalloc(&d_work, (size_t)std::max(lwork, 1) * 8) != cudaSuccess || cudaMalloc(&d_info, 4) != cudaSuccess) {
        cleanup(); if (d_work) cudaFree(d_work); h->err = "workspace allocation failed"; return ADMM_ENOMEM;
    }
    int info1 = 0, info2 = 0;
    cusolverStatus_t s1 = cusolverDnDpotrf(cs, CUBLAS_FILL_MODE_LOWER, (int)n, h->d_Sinv, (int)n, d_work, lwork, d_info);
    cudaMemcpyAsync(&info1, d_info, 4, cudaMemcpyDeviceToHost, st); cudaStreamSynchronize(st);
    cusolverStatus_t s2 = CUSOLVER_STATUS_SUCCESS;
    if (s1 == CUSOLVER_STATUS_SUCCESS && info1 == 0) {
        s2 = cusolverDnDpotri(cs, CUBLAS_FILL_MODE_LOWER, (int)n, h->d_Sinv, (int)n, d_work, lwork, d_info);
        cudaMemcpyAsync(&info2, d_info, 4, cudaMemcpyDeviceToHost, st); cudaStreamSynchronize(st);
    }
    cudaFree(d_work); cudaFree(d_info);
    cleanup();
    if (s1 != CUSOLVER_STATUS_SUCCESS || s2 != CUSOLVER_STATUS_SUCCESS) { h->err = "cuSOLVER potrf/potri failed"; return ADMM_ECUDA; }
    if (info1 != 0 || info2 != 0) { h->err = "S = I + A A^T is not positive definite (non-finite Phi?)"; return ADMM_ENOTSPD; }
    launch_symmetrize(h->d_Sinv, n, st);
    h->lds = round_up(n, 2);
    if (h->lds != n) {               // odd n: re-pitch so every row starts 16-byte aligned (K2b stages it with cp.async)
        double* padded = nullptr;
        ST_TRY(dev_alloc(h, &padded, n * h->lds));
        CU_TRY(h, cudaMemsetAsync(padded, 0, (size_t)n * h->lds * 8, st));
        CU_TRY(h, cudaMemcpy2DAsync(padded, (size_t)h->lds * 8, h->d_Sinv, (size_t)n * 8, (size_t)n * 8, (size_t)n, cudaMemcpyDeviceToDevice, st));
        CU_TRY(h, cudaStreamSynchronize(st));
        cudaFree(h->d_Sinv);
        h->d_Sinv = padded;
    }
    h->h_R.resize(n);
    CU_TRY(h, cudaMemcpyAsync(h->h_R.data(), h->d_R, (size_t)n * 8, cudaMemcpyDeviceToHost, st));
    CU_TRY(h, cudaStreamSynchronize(st));
    {   // b_hat = R o bot_rows * w_BOT (Eq. 13); the option's host pointer is not kept
        std::vector<double> bot((size_t)n, 1.0), rb((size_t)n);
        if (h->opt.bot_rows) for (int64_t j = 0; j < n; ++j) bot[j] = h->opt.bot_rows[j] ? 1.0 : 0.0;
        for (int64_t j = 0; j < n; ++j) rb[j] = h->h_R[j] * bot[j];
        ST_TRY(dev_alloc(h, &h->d_Rb, n));
        ST_TRY(dev_alloc(h, &h->d_bot, n));
        CU_TRY(h, cudaMemcpy(h->d_Rb, rb.data(), (size_t)n * 8, cudaMemcpyHostToDevice));
        CU_TRY(h, cudaMemcpy(h->d_bot, bot.data(), (size_t)n * 8, cudaMemcpyHostToDevice));
        h->opt.bot_rows = nullptr;
    }
    const double t3 = now_ms();

    // ---- work decomposition of the two contractions
    ST_TRY(tc_init(h));
    std::vector<TcUnit> u; std::vector<int32_t> b, msb;
    build_units_k3(N, n, h->sm_count, h->kblk, u, b);
    h->grid_k3 = (int)b.size() - 1;
    ST_TRY(dev_alloc(h, &h->d_units_k3, (int64_t)u.size()));
    ST_TRY(dev_alloc(h, &h->d_cta_begin_k3, (int64_t)b.size()));
    CU_TRY(h, cudaMemcpy(h->d_units_k3, u.data(), u.size() * sizeof(TcUnit), cudaMemcpyHostToDevice));
    CU_TRY(h, cudaMemcpy(h->d_cta_begin_k3, b.data(), b.size() * 4, cudaMemcpyHostToDevice));
    if (h->opt.kernel_path == ADMM_PATH_TCGEN05) {
        build_units_k1(N, n, h->sm_count, h->kblk, h->opt.storage == ADMM_STORAGE_FP32_3XTF32 ? 96 : kMaxMmaN, h->opt.k1_slab_kb, u, b, msb);
        h->grid_k1 = (int)b.size() - 1;
        h->slots_k1 = msb.back();
    } else {
        const int m_tiles = (int)cdiv(n, kTileM);
        const int splits = h->opt.storage == ADMM_STORAGE_CSR ? (int)std::max<int64_t>(1, std::min<int64_t>(32, N / 8192)) :
                           (int)std::max<int64_t>(1, std::min<int64_t>(64, (2 * h->sm_count) / std::max<int64_t>(1, cdiv(n, 64))));
        msb.resize(m_tiles + 1);
        for (int i = 0; i <= m_tiles; ++i) msb[i] = i * splits;
        h->slots_k1 = m_tiles * splits; h->grid_k1 = splits;     // grid_k1 carries the split count on the SIMT path
        u.assign(1, TcUnit{}); b.assign(2, 0);
    }
    ST_TRY(dev_alloc(h, &h->d_units_k1, (int64_t)u.size()));
    ST_TRY(dev_alloc(h, &h->d_cta_begin_k1, (int64_t)b.size()));
    ST_TRY(dev_alloc(h, &h->d_mtile_slot_begin, (int64_t)msb.size()));
    CU_TRY(h, cudaMemcpy(h->d_units_k1, u.data(), u.size() * sizeof(TcUnit), cudaMemcpyHostToDevice));
    CU_TRY(h, cudaMemcpy(h->d_cta_begin_k1, b.data(), b.size() * 4, cudaMemcpyHostToDevice));
    CU_TRY(h, cudaMemcpy(h->d_mtile_slot_begin, msb.data(), msb.size() * 4, cudaMemcpyHostToDevice));

    h->ms[0] = t1 - t0; h->ms[1] = t2 - t1; h->ms[2] = t3 - t2; h->ms[3] = now_ms() - t0;
    return ADMM_OK;
}

admm_status admm_setup(admm_handle** out, const float* phi, int32_t phi_on_device, int64_t N, int64_t n, int64_t ld,
                       const uint8_t* point_class, const admm_class* classes, int32_t n_classes, const admm_options* opt) {
    if (!out) { g_setup_err = "out is NULL"; return ADMM_EINVAL; }
    *out = nullptr;
    if (!phi || !point_class || !classes) { g_setup_err = "phi / point_class / classes is NULL"; return ADMM_EINVAL; }
    if (N < 1 || n < 1 || ld < n) { g_setup_err = "need N >= 1, n >= 1, ld >= n"; return ADMM_EINVAL; }
    if (N >= (1ll << 31) - 256 || n >= (1ll << 31) - 256) { g_setup_err = "N, n must fit 32-bit tile coordinates"; return ADMM_EINVAL; }
    if (n_classes < 1 || n_classes > kMaxClasses) { g_setup_err = "n_classes must be in [1, 8]"; return ADMM_EINVAL; }
    for (int k = 0; k < n_classes; ++k) {
        if (classes[k].sense != 1 && classes[k].sense != -1) { g_setup_err = "class sense must be +1 or -1"; return ADMM_EINVAL; }
        if (!(classes[k].threshold > 0.f) || !std::isfinite(classes[k].threshold)) { g_setup_err = "class threshold must be finite and > 0"; return ADMM_EINVAL; }
        if (classes[k].hard < 0 || classes[k].hard > 2) { g_setup_err = "class hard must be 0, 1 or 2"; return ADMM_EINVAL; }
        if (classes[k].hard == 2 && classes[k].threshold != 1.f) { g_setup_err = "a homogeneous hard class (hard = 2) must have threshold 1"; return ADMM_EINVAL; }
    }
    admm_options o;
    if (opt) o = *opt; else admm_default_options(&o);
    if (o.check_every <= 0) o.check_every = 10;
    if (!(o.eps_abs > 0.f)) o.eps_abs = 1e-6f;
    if (o.storage < ADMM_STORAGE_FP32_3XTF32 || o.storage > ADMM_STORAGE_CSR) { g_setup_err = "unknown storage mode"; return ADMM_EINVAL; }
    if (o.compaction != 1) { g_setup_err = "compaction must be 1 (masking without compaction is not offered)"; return ADMM_EINVAL; }
    if (o.bot_rows) for (int64_t j = 0; j < n; ++j)
        if (o.bot_rows[j] > 1) { g_setup_err = "bot_rows entries must be 0 or 1"; return ADMM_EINVAL; }
    if (o.dose_only != 0 && o.dose_only != 1) { g_setup_err = "dose_only must be 0 or 1"; return ADMM_EINVAL; }
    if (!(o.warm_start_ratio >= 0.f) || !std::isfinite(o.warm_start_ratio)) { g_setup_err = "warm_start_ratio must be finite and >= 0"; return ADMM_EINVAL; }
    if (o.warm_start_ratio > 0.f && o.warm_start_ratio < 1.f) { g_setup_err = "warm_start_ratio, if set, must be >= 1"; return ADMM_EINVAL; }
    if (o.dose_only && o.storage == ADMM_STORAGE_CSR) { g_setup_err = "dose_only is not offered with ADMM_STORAGE_CSR"; return ADMM_EINVAL; }
    if (o.storage == ADMM_STORAGE_CSR) {
        // sparse contractions run on the plain FP32 ALUs with the orchestration of the cross-check path
        o.kernel_path = ADMM_PATH_SIMT;
        if (!(o.csr_rel_threshold > 0.f)) o.csr_rel_threshold = 1e-3f;
        if (!(o.csr_rel_threshold < 1.f)) { g_setup_err = "csr_rel_threshold must be in (0, 1)"; return ADMM_EINVAL; }
    }
    if (o.storage == ADMM_STORAGE_BF16 && o.kernel_path != ADMM_PATH_TCGEN05) {
        g_setup_err = "ADMM_STORAGE_BF16 exists on the tcgen05 path only"; return ADMM_EINVAL;
    }
    if (o.kernel_path != ADMM_PATH_TCGEN05 && o.kernel_path != ADMM_PATH_SIMT) { g_setup_err = "unknown kernel_path"; return ADMM_EINVAL; }
    admm_handle* h = new (std::nothrow) admm_handle();
    if (!h) { g_setup_err = "host allocation failed"; return ADMM_ENOMEM; }
    h->opt = o;
    admm_status s = setup_impl(h, phi, phi_on_device, N, n, ld, point_class, classes, n_classes);
    if (s != ADMM_OK) {
        g_setup_err = h->err;
        cudaGetLastError();
        free_all(h);
        delete h;
        return s;
    }
    *out = h;
    return ADMM_OK;
}

}  // extern "C"

static admm_status ensure_batch_buffers(admm_handle* h, int B) {
    const int Bpad = (int)round_up(B, 16);
    if (Bpad <= h->Bpad && h->d_s1) return ADMM_OK;
    // the epilogues address [slot][ldN] arrays with 32-bit element offsets
    if ((int64_t)Bpad * h->ldN >= (1ll << 32)) { h->err = "B * N too large: the batch arrays must hold fewer than 2^32 elements"; return ADMM_EINVAL; }
    const bool simt = h->opt.kernel_path == ADMM_PATH_SIMT;
    h->map_cache.clear();
    h->Bpad = 0;
    h->k2_rows = k2_choose_rows(h, Bpad);
    ST_TRY(dev_alloc(h, &h->d_s1, (int64_t)Bpad * h->ldN));
    ST_TRY(dev_alloc(h, &h->d_ghi, 2 * (int64_t)Bpad * h->ldN));          // hi plane, then lo plane
    h->d_glo = h->d_ghi + (int64_t)Bpad * h->ldN;
    ST_TRY(dev_alloc(h, &h->d_s2, (int64_t)Bpad * h->ldn));
    ST_TRY(dev_alloc(h, &h->d_rhs, (int64_t)Bpad * h->ldn));
    CU_TRY(h, cudaMemsetAsync(h->d_rhs, 0, (size_t)Bpad * h->ldn * 8, h->stream));   // pad columns are read (x 0) by K2b
    ST_TRY(dev_alloc(h, &h->d_vhi, 2 * (int64_t)Bpad * h->ldn));
    h->d_vlo = h->d_vhi + (int64_t)Bpad * h->ldn;
    ST_TRY(dev_alloc(h, &h->d_partial, (int64_t)h->slots_k1 * std::min(Bpad, max_pass(h)) * kTileM));
    const int grid1 = simt ? (int)cdiv(h->N, 128) : h->grid_k3;
    ST_TRY(dev_alloc(h, &h->d_resid1, (int64_t)grid1 * kMaxBpad * kNumResid));
    ST_TRY(dev_alloc(h, &h->d_resid2, (int64_t)k2b_grid(h, Bpad) * kMaxBpad * kNumResid));
    ST_TRY(dev_alloc(h, &h->d_hinge, (int64_t)grid1 * kMaxBpad * kMaxClasses));
    ST_TRY(dev_alloc(h, &h->d_slot_plan, Bpad));
    ST_TRY(dev_alloc(h, &h->d_utab, kMaxClasses * kMaxBpad));
    ST_TRY(dev_alloc(h, &h->d_crtab, kMaxClasses * kMaxBpad));
    ST_TRY(dev_alloc(h, &h->d_beta, kMaxBpad));
    ST_TRY(dev_alloc(h, &h->d_rho, kMaxBpad));
    ST_TRY(dev_alloc(h, &h->d_wnorm, (int64_t)kMaxBpad * kMaxClasses));
    ST_TRY(dev_alloc(h, &h->d_active_counts, (int64_t)Bpad * kMaxClasses));
    ST_TRY(dev_alloc(h, &h->d_conv_flags, Bpad));
    ST_TRY(dev_alloc(h, &h->d_bact, 1));
    ST_TRY(dev_alloc(h, &h->d_moves, Bpad));
    ST_TRY(dev_alloc(h, &h->d_nmoves, 1));
    ST_TRY(dev_alloc(h, &h->d_iters_plan, Bpad));
    ST_TRY(dev_alloc(h, &h->d_res_plan, 2 * Bpad));
    ST_TRY(dev_alloc(h, &h->d_t_f32, (int64_t)Bpad * h->ldn));
    ST_TRY(dev_alloc(h, &h->d_obj, kMaxBpad));
    ST_TRY(dev_alloc(h, &h->d_plan_slot, Bpad));
    ST_TRY(dev_alloc(h, &h->d_tout, (int64_t)Bpad * h->n));
    if (simt) ST_TRY(dev_alloc(h, &h->d_qbuf, (int64_t)std::min(Bpad, max_pass(h)) * h->ldN));
    if (!h->h_bact_ring) {
        CU_TRY(h, cudaHostAlloc(reinterpret_cast<void**>(&h->h_bact_ring), 8 * sizeof(int32_t), cudaHostAllocDefault));
        for (auto& e : h->bact_ev) CU_TRY(h, cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
    }
    h->Bpad = Bpad;
    return ADMM_OK;
}

namespace {
struct SlotTables {
    std::vector<float> utab, crtab;         // [kMaxClasses][kMaxBpad]
    std::vector<double> beta, rho, wnorm;   // [kMaxBpad], [kMaxBpad][kMaxClasses]
};
admm_status upload_tables(admm_handle* h, const SlotTables& T) {
    cudaStream_t st = h->stream;
    CU_TRY(h, cudaMemcpyAsync(h->d_utab, T.utab.data(), T.utab.size() * 4, cudaMemcpyHostToDevice, st));
    CU_TRY(h, cudaMemcpyAsync(h->d_crtab, T.crtab.data(), T.crtab.size() * 4, cudaMemcpyHostToDevice, st));
    CU_TRY(h, cudaMemcpyAsync(h->d_beta, T.beta.data(), T.beta.size() * 8, cudaMemcpyHostToDevice, st));
    CU_TRY(h, cudaMemcpyAsync(h->d_rho, T.rho.data(), T.rho.size() * 8, cudaMemcpyHostToDevice, st));
    CU_TRY(h, cudaMemcpyAsync(h->d_slot_plan, h->slot_plan.data(), h->slot_plan.size() * 4, cudaMemcpyHostToDevice, st));
    CU_TRY(h, cudaMemcpyAsync(h->d_wnorm, T.wnorm.data(), T.wnorm.size() * 8, cudaMemcpyHostToDevice, st));
    return ADMM_OK;
}
// The live count after each check travels to the host through a small ring of pinned words + events.  The host never waits for the
// check it has just enqueued: it waits for the one before, so a whole check interval of work is always queued behind the GPU and
// the launch sizes (n_mma, grids) follow the device's live count with a lag of at most one interval.
struct LiveCount {
    admm_handle* h; int head = 0, tail = 0;        // ring entries [tail, head) are in flight
    admm_status push() {
        const int e = head % 8;
        CU_TRY(h, cudaMemcpyAsync(h->h_bact_ring + e, h->d_bact, 4, cudaMemcpyDeviceToHost, h->stream));
        CU_TRY(h, cudaEventRecord(h->bact_ev[e], h->stream));
        ++head;
        return ADMM_OK;
    }
    // waits until at most `keep` copies are still in flight; returns the newest value that has arrived (or `cur`)
    admm_status drain(int keep, int* cur) {
        while (head - tail > keep) {
            const int e = tail % 8;
            CU_TRY(h, cudaEventSynchronize(h->bact_ev[e]));
            *cur = std::min(*cur, (int)h->h_bact_ring[e]);
            ++tail;
        }
        while (head > tail && cudaEventQuery(h->bact_ev[tail % 8]) == cudaSuccess) {
            *cur = std::min(*cur, (int)h->h_bact_ring[tail % 8]);
            ++tail;
        }
        return ADMM_OK;
    }
};
}  // namespace

extern "C" {

admm_status admm_solve_batch(admm_handle* h, int32_t B, const float* weights, const float* rho, const uint32_t* row_mask,
                             float tol, int32_t max_iter, int32_t fixed_iters, float* t_out, double* obj_out,
                             float* res_out, int32_t* iters_out) {
    if (!h) return ADMM_EINVAL;
    if (h->opt.dose_only) { h->err = "this handle was made with dose_only = 1: it only serves admm_dose"; return ADMM_ESTATE; }
    if (!weights) { h->err = "weights is NULL"; return ADMM_EINVAL; }
    if (B < 1 || B > kMaxBpad - 16) { h->err = "B must be in [1, 496]"; return ADMM_EINVAL; }
    if (fixed_iters < 0) { h->err = "fixed_iters < 0"; return ADMM_EINVAL; }
    if (fixed_iters == 0 && (!(tol > 0.f) || max_iter < 1)) { h->err = "need tol > 0 and max_iter >= 1 (or fixed_iters > 0)"; return ADMM_EINVAL; }
    const int K = h->n_classes, W = K + 1;
    for (int64_t i = 0; i < (int64_t)B * W; ++i)
        if (!(weights[i] >= 0.f) || !std::isfinite(weights[i])) { h->err = "weights must be finite and >= 0"; return ADMM_EINVAL; }
    if (rho) for (int p = 0; p < B; ++p)
        if (!(rho[p] > 0.f) || !std::isfinite(rho[p])) { h->err = "rho must be finite and > 0"; return ADMM_EINVAL; }
    CU_TRY(h, cudaSetDevice(h->opt.device));
    cudaStream_t st = h->stream;
    const double wall0 = now_ms();
    h->launch_count = 0; h->ktimes = KernelTimes{}; h->plan_iters = 0; h->solved = false; h->presolved = 0;
    ST_TRY(ensure_batch_buffers(h, B));
    h->B = B;
    const bool simt = h->opt.kernel_path == ADMM_PATH_SIMT;
    const int total_iters = fixed_iters > 0 ? fixed_iters : max_iter;
    const int check_every = h->opt.check_every;

    // ---- row masks and active counts N_{k,p}
    h->mask_words = cdiv(h->N, 32);
    h->has_mask = row_mask != nullptr;
    if (row_mask) {
        if ((int64_t)B * h->mask_words > h->mask_capacity) {
            ST_TRY(dev_alloc(h, &h->d_mask, (int64_t)B * h->mask_words));
            h->mask_capacity = (int64_t)B * h->mask_words;
        }
        CU_TRY(h, cudaMemcpyAsync(h->d_mask, row_mask, (size_t)B * h->mask_words * 4,
                                  is_device_ptr(row_mask) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st));
    }
    launch_count_active(row_mask ? h->d_mask : nullptr, h->mask_words, h->d_point_class, h->N, B, h->d_active_counts, st);
    std::vector<int32_t> counts((size_t)B * kMaxClasses);
    CU_TRY(h, cudaMemcpyAsync(counts.data(), h->d_active_counts, counts.size() * 4, cudaMemcpyDeviceToHost, st));
    CU_TRY(h, cudaStreamSynchronize(st));

    // ---- per-slot tables (slot == plan at the start)
    SlotTables T;
    T.utab.assign((size_t)kMaxClasses * kMaxBpad, 0.f); T.crtab.assign((size_t)kMaxClasses * kMaxBpad, 0.f);
    T.beta.assign(kMaxBpad, 0.0); T.rho.assign(kMaxBpad, 1.0); T.wnorm.assign((size_t)kMaxBpad * kMaxClasses, 0.0);
    h->slot_plan.assign(h->Bpad, 0); h->plan_slot.assign(B, 0); h->iters.assign(B, 0);
    int64_t n_min_class = h->class_count[0];
    for (int k = 1; k < K; ++k) n_min_class = std::min(n_min_class, h->class_count[k]);
    bool box_optimum_finite = true;           // presolve needs a finite box optimum: no hard class with c < 0
    for (int k = 0; k < K; ++k) if (h->classes[k].hard == 1 && h->classes[k].sense > 0) box_optimum_finite = false;   // c < 0 with u = infinity
    for (int p = 0; p < B; ++p) {
        const double beta = weights[(size_t)p * W + K];
        // default: (kappa / N_min) sqrt(beta0 / max(beta, beta0/floor)), kappa = 1, beta0 = 0.05 (reading R8)
        const double r = rho ? (double)rho[p] : (1.0 / (double)n_min_class) * std::sqrt(0.05 / std::max(beta, 0.05 / kRhoFloorDiv));
        T.beta[p] = beta; T.rho[p] = r;
        for (int k = 0; k < K; ++k) {
            const double Nk = (double)h->class_count[k], Nkp = (double)counts[(size_t)p * kMaxClasses + k];
            const double wk = weights[(size_t)p * W + k], thr = h->classes[k].threshold, sense = h->classes[k].sense;
            // u_hat = u / D = (w thr / N_kp) * N_k ;  c_hat / rho = (-sense / N_k) / rho ;  hard class: u = infinity (Eq. 15)
            float uh = (float)(Nkp > 0 ? wk * thr * Nk / Nkp : 0.0);
            if (h->classes[k].hard) uh = Nkp > 0 ? INFINITY : 0.f;
            T.utab[(size_t)k * kMaxBpad + p] = uh;
            T.crtab[(size_t)k * kMaxBpad + p] = h->classes[k].hard == 2 ? 0.f : (float)((-sense / Nk) / r);   // c = 0 for a homogeneous hard class
            T.wnorm[(size_t)p * kMaxClasses + k] = (Nkp > 0 && !h->classes[k].hard) ? wk / Nkp : 0.0;
        }
        h->slot_plan[p] = p; h->plan_slot[p] = p;
    }
    ST_TRY(upload_tables(h, T));
    const int32_t B32 = B;
    CU_TRY(h, cudaMemcpyAsync(h->d_bact, &B32, 4, cudaMemcpyHostToDevice, st));
    launch_init_plan_records(h, B, st);

    // ---- zero start (R6) and the first K1 operand
    CU_TRY(h, cudaMemsetAsync(h->d_s1, 0, (size_t)h->Bpad * h->ldN * 4, st));
    CU_TRY(h, cudaMemsetAsync(h->d_ghi, 0, (size_t)h->Bpad * h->ldN * 4, st));
    CU_TRY(h, cudaMemsetAsync(h->d_glo, 0, (size_t)h->Bpad * h->ldN * 4, st));
    CU_TRY(h, cudaMemsetAsync(h->d_s2, 0, (size_t)h->Bpad * h->ldn * 8, st));
    CU_TRY(h, cudaMemsetAsync(h->d_vhi, 0, (size_t)h->Bpad * h->ldn * 4, st));
    CU_TRY(h, cudaMemsetAsync(h->d_vlo, 0, (size_t)h->Bpad * h->ldn * 4, st));
    float* qbuf = h->d_qbuf;     // SIMT path only: Q [pass][ldN]

    Profiler prof; prof.on = h->opt.profile_kernels != 0;
    cudaEvent_t ev0, ev1, ev2;
    cudaEventCreate(&ev0); cudaEventCreate(&ev1); cudaEventCreate(&ev2);
    struct EvGuard { cudaEvent_t a, b, c; ~EvGuard() { cudaEventDestroy(a); cudaEventDestroy(b); cudaEventDestroy(c); } } evg{ev0, ev1, ev2};
    cudaEventRecord(ev0, st);

    int Bact = B;                       // the HOST's upper bound on the live count; the device's own is *d_bact
    LiveCount live{h};
    EpiParams ep0 = base_epi(h); ep0.slot0 = 0; ep0.n_slots_active = B;

    // ---- presolve (deviation D1): plans whose box optimum is feasible are solved in closed form (t* = 0)
    if (fixed_iters == 0 && h->opt.presolve && box_optimum_finite) {
        launch_presolve_state(ep0, B, st);
        launch_emit_g(ep0, B, st);
        for (int s0 = 0; s0 < B; s0 += max_pass(h)) {
            const int nact = std::min(max_pass(h), B - s0);
            const int n_mma = (int)round_up(nact, 16);
            if (simt) launch_simt_k1(h, s0, nact, n_mma, h->grid_k1, st);
            else ST_TRY(contract(h, EPI_K1_PARTIAL, s0, nact, h->d_ghi, h->d_glo, false));
            launch_presolve_test(h, s0, nact, n_mma, 1e-5, st);
        }
        launch_presolve_reset(h, B, st);
        h->launch_count += 4;
        launch_compaction(h, Bact, st);
        ST_TRY(live.push());
        ST_TRY(live.drain(0, &Bact));
        h->presolved = B - Bact;
    }
    if (Bact > 0) { ep0.n_slots_active = Bact; launch_emit_g(ep0, Bact, st); h->launch_count++; }

    const int grid1 = simt ? (int)cdiv(h->N, 128) : h->grid_k3;
    int it = 0;
    while (it < total_iters && Bact > 0) {
        ++it;
        const bool check = (fixed_iters > 0) ? (it == total_iters) : (it % check_every == 0 || it == total_iters);
        // ---- K1 + K2a per pass of plans: rhs = R o (Phi^T G) - (2 z2 - s2)
        for (int s0 = 0; s0 < Bact; s0 += max_pass(h)) {
            const int nact = std::min(max_pass(h), Bact - s0);
            const int n_mma = (int)round_up(nact, 16);
            prof.begin(h, 0);
            if (simt) launch_simt_k1(h, s0, nact, n_mma, h->grid_k1, st);
            else ST_TRY(contract(h, EPI_K1_PARTIAL, s0, nact, h->d_ghi, h->d_glo, false, nullptr, true));
            prof.end(h);
            prof.begin(h, 1);
            launch_k2a(h, s0, nact, n_mma, st);
            prof.end(h);
        }
        // ---- K2b: v = S^-1 rhs, epilogue-2
        prof.begin(h, 1);
        launch_k2b(h, Bact, check, st);
        prof.end(h);
        // ---- K3: Q = Phi (R o v), epilogue-1
        for (int s0 = 0; s0 < Bact; s0 += max_pass(h)) {
            const int nact = std::min(max_pass(h), Bact - s0);
            prof.begin(h, 2);
            if (simt) {
                EpiParams ep = base_epi(h);
                ep.slot0 = s0; ep.n_slots_active = nact; ep.n_mma = (int)round_up(nact, 16);
                ep.bact_dev = h->d_bact;
                ep.resid_partial = check ? h->d_resid1 : nullptr;
                launch_simt_k3(h, ep, EPI_K3_STATE, h->d_vhi + (int64_t)s0 * h->ldn, h->d_vlo + (int64_t)s0 * h->ldn, qbuf, st);
            } else {
                ST_TRY(contract(h, EPI_K3_STATE, s0, nact, h->d_vhi, h->d_vlo, check, nullptr, true));
            }
            prof.end(h);
        }
        if (!check) continue;
        // ---- H5: stopping rule on the device, then (tolerance mode) compaction on the device
        prof.begin(h, 3);
        launch_convergence(h, Bact, grid1, k2b_grid(h, Bact), fixed_iters > 0 ? 0.f : tol, h->opt.eps_abs, it, st);
        if (fixed_iters == 0) launch_compaction(h, Bact, st);
        prof.end(h);
        if (fixed_iters == 0) {
            ST_TRY(live.push());
            ST_TRY(live.drain(1, &Bact));           // wait for the PREVIOUS check only: the GPU always has an interval queued
        }
        if (cudaGetLastError() != cudaSuccess) { h->err = "a hot-path kernel failed to launch"; return ADMM_ECUDA; }
    }
    ST_TRY(live.drain(0, &Bact));
    cudaEventRecord(ev1, st);

    // ---- H6: t = rho R y2, objective P(t) through one more Phi contraction (all B slots, frozen ones included)
    float *t_hi = h->d_vhi, *t_lo = h->d_vlo;          // v operands are dead now: reuse as the T operand
    float* t_f32 = h->d_t_f32;
    launch_make_t(h, B, t_hi, t_lo, t_f32, st);
    for (int s0 = 0; s0 < B; s0 += max_pass(h)) {
        const int nact = std::min(max_pass(h), B - s0);
        if (simt) {
            EpiParams ep = base_epi(h);
            ep.slot0 = s0; ep.n_slots_active = nact; ep.n_mma = (int)round_up(nact, 16);
            launch_simt_k3(h, ep, EPI_OBJECTIVE, t_hi + (int64_t)s0 * h->ldn, t_lo + (int64_t)s0 * h->ldn, qbuf, st);
        } else {
            ST_TRY(contract(h, EPI_OBJECTIVE, s0, nact, t_hi, t_lo, false));
        }
    }
    launch_objective_reduce(h, B, grid1, t_f32, h->d_wnorm, h->d_obj, st);
    cudaEventRecord(ev2, st);

    // ---- read back what the host needs; nothing of the caller's is written until everything has succeeded
    std::vector<double> obj_slot(B);
    std::vector<float> res_plan((size_t)2 * B);
    CU_TRY(h, cudaMemcpyAsync(h->slot_plan.data(), h->d_slot_plan, (size_t)B * 4, cudaMemcpyDeviceToHost, st));
    CU_TRY(h, cudaMemcpyAsync(obj_slot.data(), h->d_obj, (size_t)B * 8, cudaMemcpyDeviceToHost, st));
    CU_TRY(h, cudaMemcpyAsync(h->iters.data(), h->d_iters_plan, (size_t)B * 4, cudaMemcpyDeviceToHost, st));
    CU_TRY(h, cudaMemcpyAsync(res_plan.data(), h->d_res_plan, (size_t)B * 8, cudaMemcpyDeviceToHost, st));
    CU_TRY(h, cudaStreamSynchronize(st));
    if (cudaGetLastError() != cudaSuccess) { h->err = "a hot-path kernel failed"; return ADMM_ECUDA; }
    prof.harvest(h);
    for (int s = 0; s < B; ++s) h->plan_slot[h->slot_plan[s]] = s;
    std::vector<double> obj_plan(B);
    for (int p = 0; p < B; ++p) obj_plan[p] = obj_slot[h->plan_slot[p]];
    // ---- outputs, in plan order
    if (t_out) {
        CU_TRY(h, cudaMemcpyAsync(h->d_plan_slot, h->plan_slot.data(), (size_t)B * 4, cudaMemcpyHostToDevice, st));
        if (is_device_ptr(t_out)) {
            launch_gather_rows(t_f32, h->ldn, h->d_plan_slot, B, h->n, t_out, st);
        } else {
            launch_gather_rows(t_f32, h->ldn, h->d_plan_slot, B, h->n, h->d_tout, st);
            CU_TRY(h, cudaMemcpyAsync(t_out, h->d_tout, (size_t)B * h->n * 4, cudaMemcpyDeviceToHost, st));
        }
        CU_TRY(h, cudaStreamSynchronize(st));
    }
    auto put = [&](void* dst, const void* src, size_t bytes) -> cudaError_t {
        if (!dst) return cudaSuccess;
        if (is_device_ptr(dst)) return cudaMemcpy(dst, src, bytes, cudaMemcpyHostToDevice);
        memcpy(dst, src, bytes); return cudaSuccess;
    };
    CU_TRY(h, put(obj_out, obj_plan.data(), (size_t)B * 8));
    CU_TRY(h, put(res_out, res_plan.data(), (size_t)B * 8));
    CU_TRY(h, put(iters_out, h->iters.data(), (size_t)B * 4));
    float ms_it = 0, ms_fin = 0;
    cudaEventElapsedTime(&ms_it, ev0, ev1); cudaEventElapsedTime(&ms_fin, ev1, ev2);
    h->ms[4] = ms_it; h->ms[5] = ms_fin; h->ms[6] = now_ms() - wall0;
    for (int p = 0; p < B; ++p) h->plan_iters += h->iters[p];
    h->solved = true;
    return ADMM_OK;
}

admm_status admm_contract_probe(admm_handle* h, int32_t which, int32_t B, const float* small, double* out) {
    if (!h || !small || !out) return ADMM_EINVAL;
    if (B < 1 || B > max_pass(h) || (which != 0 && which != 1)) { h->err = "probe: need 1 <= B <= 96 (fp32 path) / 256, which in {0,1}"; return ADMM_EINVAL; }
    if (h->opt.dose_only && which == 0) { h->err = "dose_only handle: no Phi^T product"; return ADMM_ESTATE; }
    CU_TRY(h, cudaSetDevice(h->opt.device));
    cudaStream_t st = h->stream;
    ST_TRY(ensure_batch_buffers(h, B));
    h->B = B; h->solved = false; h->has_mask = false;
    const bool simt = h->opt.kernel_path == ADMM_PATH_SIMT;
    const int64_t K = which == 0 ? h->N : h->n, ldK = which == 0 ? h->ldN : h->ldn;
    const int64_t rows = which == 0 ? h->n : h->N;
    float* hi = which == 0 ? h->d_ghi : h->d_vhi; float* lo = which == 0 ? h->d_glo : h->d_vlo;
    float* stage = nullptr; double* dout = nullptr; float* qbuf = nullptr;
    struct G { void* a; void* b; void* c; ~G() { if (a) cudaFree(a); if (b) cudaFree(b); if (c) cudaFree(c); } } g{nullptr, nullptr, nullptr};
    ST_TRY(dev_alloc(h, &stage, (int64_t)h->Bpad * ldK)); g.a = stage;
    CU_TRY(h, cudaMemsetAsync(stage, 0, (size_t)h->Bpad * ldK * 4, st));
    CU_TRY(h, cudaMemcpy2DAsync(stage, (size_t)ldK * 4, small, (size_t)K * 4, (size_t)K * 4, (size_t)B, cudaMemcpyHostToDevice, st));
    launch_split_small(stage, (int64_t)h->Bpad * ldK, ldK, hi, lo, h->opt.storage == ADMM_STORAGE_BF16, st);
    const int n_mma = (int)round_up(B, 16);
    if (which == 0) {
        if (simt) launch_simt_k1(h, 0, B, n_mma, h->grid_k1, st);
        else ST_TRY(contract(h, EPI_K1_PARTIAL, 0, B, hi, lo, false));
        ST_TRY(dev_alloc(h, &dout, (int64_t)B * h->n)); g.b = dout;
        launch_reduce_partial(h, B, n_mma, dout, st);
        CU_TRY(h, cudaMemcpyAsync(out, dout, (size_t)B * h->n * 8, cudaMemcpyDeviceToHost, st));
        CU_TRY(h, cudaStreamSynchronize(st));
    } else {
        ST_TRY(dev_alloc(h, &qbuf, (int64_t)h->Bpad * h->ldN)); g.c = qbuf;
        if (simt) {
            EpiParams ep = base_epi(h); ep.slot0 = 0; ep.n_slots_active = B; ep.n_mma = n_mma;
            launch_simt_k3(h, ep, EPI_RAW, hi, lo, qbuf, st);
        } else {
            ST_TRY(contract_raw(h, B, hi, lo, qbuf));
        }
        std::vector<float> tmp((size_t)B * h->ldN);
        CU_TRY(h, cudaMemcpyAsync(tmp.data(), qbuf, tmp.size() * 4, cudaMemcpyDeviceToHost, st));
        CU_TRY(h, cudaStreamSynchronize(st));
        for (int p = 0; p < B; ++p) for (int64_t i = 0; i < rows; ++i) out[(int64_t)p * rows + i] = tmp[(size_t)p * h->ldN + i];
    }
    return ADMM_OK;
}

// Dose calculation between the passes of II.C: dose[p][i] = Phi_i . t_p through the K3 contraction.
// Leaves the dose in h->d_s1 [Bpad][ldN] (the state of the last solve is given up).
static admm_status dose_into_s1(admm_handle* h, int32_t B, const float* t, int64_t ld_t) {
    if (!t) { h->err = "t is NULL"; return ADMM_EINVAL; }
    if (B < 1 || B > kMaxBpad - 16) { h->err = "B must be in [1, 496]"; return ADMM_EINVAL; }
    if (ld_t < h->n) { h->err = "ld_t < n"; return ADMM_EINVAL; }
    if (h->opt.storage == ADMM_STORAGE_CSR) { h->err = "admm_dose is not offered with ADMM_STORAGE_CSR"; return ADMM_EINVAL; }
    CU_TRY(h, cudaSetDevice(h->opt.device));
    cudaStream_t st = h->stream;
    ST_TRY(ensure_batch_buffers(h, B));
    h->B = B; h->solved = false; h->has_mask = false;
    const bool simt = h->opt.kernel_path == ADMM_PATH_SIMT;
    // stage T [Bpad][ldn] (rows >= B and the pad columns are zero), split into the hi / lo operand pair of the storage mode
    float* stage = h->d_t_f32;                       // [Bpad][ldn] scratch of the finalise step
    CU_TRY(h, cudaMemsetAsync(stage, 0, (size_t)h->Bpad * h->ldn * 4, st));
    CU_TRY(h, cudaMemcpy2DAsync(stage, (size_t)h->ldn * 4, t, (size_t)ld_t * 4, (size_t)h->n * 4, (size_t)B,
                                is_device_ptr(t) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st));
    launch_split_small(stage, (int64_t)h->Bpad * h->ldn, h->ldn, h->d_vhi, h->d_vlo, h->opt.storage == ADMM_STORAGE_BF16, st);
    float* q = h->d_s1;
    for (int s0 = 0; s0 < B; s0 += max_pass(h)) {
        const int nact = std::min(max_pass(h), B - s0);
        if (simt) {
            EpiParams ep = base_epi(h); ep.slot0 = s0; ep.n_slots_active = nact; ep.n_mma = (int)round_up(nact, 16);
            launch_simt_k3(h, ep, EPI_RAW, h->d_vhi + (int64_t)s0 * h->ldn, h->d_vlo + (int64_t)s0 * h->ldn, q + (int64_t)s0 * h->ldN, st);
        } else {
            ST_TRY(contract(h, EPI_RAW, s0, nact, h->d_vhi, h->d_vlo, false, q));
        }
    }
    return ADMM_OK;
}
static admm_status copy_dose_out(admm_handle* h, int32_t B, float* dose_out) {
    CU_TRY(h, cudaMemcpy2DAsync(dose_out, (size_t)h->N * 4, h->d_s1, (size_t)h->ldN * 4, (size_t)h->N * 4, (size_t)B,
                                is_device_ptr(dose_out) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, h->stream));
    return ADMM_OK;
}

admm_status admm_dose(admm_handle* h, int32_t B, const float* t, int64_t ld_t, float* dose_out) {
    if (!h) return ADMM_EINVAL;
    if (!dose_out) { h->err = "dose_out is NULL"; return ADMM_EINVAL; }
    ST_TRY(dose_into_s1(h, B, t, ld_t));
    ST_TRY(copy_dose_out(h, B, dose_out));
    CU_TRY(h, cudaStreamSynchronize(h->stream));
    if (cudaGetLastError() != cudaSuccess) { h->err = "admm_dose: a kernel failed"; return ADMM_ECUDA; }
    return ADMM_OK;
}

// Second-pass low-dose volumes of all plans (PAPER.md II.C.1, :110-114) from their first-pass dose on this handle's points.
admm_status admm_lowdose_volumes(admm_handle* h, int32_t B, const float* t, int64_t ld_t, float d_lo, float d_hi,
                                 uint32_t* in_volume, uint32_t* any_volume, float* dose_out) {
    if (!h) return ADMM_EINVAL;
    if (!in_volume) { h->err = "in_volume is NULL"; return ADMM_EINVAL; }
    if (!(d_lo < d_hi) || !std::isfinite(d_lo) || !std::isfinite(d_hi)) { h->err = "need finite d_lo < d_hi"; return ADMM_EINVAL; }
    ST_TRY(dose_into_s1(h, B, t, ld_t));
    cudaStream_t st = h->stream;
    const int64_t words = cdiv(h->N, 32);
    uint32_t* d_in = nullptr; uint32_t* d_any = nullptr;
    struct G { uint32_t*& a; uint32_t*& b; ~G() { if (a) cudaFree(a); if (b) cudaFree(b); } } g{d_in, d_any};
    ST_TRY(dev_alloc(h, &d_in, (int64_t)B * words));
    ST_TRY(dev_alloc(h, &d_any, words));
    CU_TRY(h, cudaMemsetAsync(d_any, 0, (size_t)words * 4, st));
    launch_lowdose_volume(h->d_s1, h->ldN, h->N, B, d_lo, d_hi, d_in, words, d_any, st);
    CU_TRY(h, cudaMemcpyAsync(in_volume, d_in, (size_t)B * words * 4, is_device_ptr(in_volume) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, st));
    if (any_volume) CU_TRY(h, cudaMemcpyAsync(any_volume, d_any, (size_t)words * 4, is_device_ptr(any_volume) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, st));
    if (dose_out) ST_TRY(copy_dose_out(h, B, dose_out));
    CU_TRY(h, cudaStreamSynchronize(st));
    if (cudaGetLastError() != cudaSuccess) { h->err = "admm_lowdose_volumes: a kernel failed"; return ADMM_ECUDA; }
    return ADMM_OK;
}

admm_status admm_get_state(admm_handle* h, int32_t plan, float* z1, float* y1, double* z2, double* y2) {
    if (!h) return ADMM_EINVAL;
    if (!h->solved) { h->err = "admm_get_state before a successful admm_solve_batch"; return ADMM_ESTATE; }
    if (plan < 0 || plan >= h->B) { h->err = "plan out of range"; return ADMM_EINVAL; }
    CU_TRY(h, cudaSetDevice(h->opt.device));
    cudaStream_t st = h->stream;
    const int slot = h->plan_slot[plan];
    float *dz1 = nullptr, *dy1 = nullptr; double *dz2 = nullptr, *dy2 = nullptr;
    struct G { void* p[4]; ~G() { for (void* q : p) if (q) cudaFree(q); } } g{{nullptr, nullptr, nullptr, nullptr}};
    auto stage = [&](auto** dev, auto* user, int64_t count, int gi) -> admm_status {
        using T = std::remove_pointer_t<std::remove_pointer_t<decltype(dev)>>;
        if (!user) { *dev = nullptr; return ADMM_OK; }
        if (is_device_ptr(user)) { *dev = user; return ADMM_OK; }
        T* tmp = nullptr;
        ST_TRY(dev_alloc(h, &tmp, count));
        g.p[gi] = tmp; *dev = tmp;
        return ADMM_OK;
    };
    ST_TRY(stage(&dz1, z1, h->N, 0)); ST_TRY(stage(&dy1, y1, h->N, 1));
    ST_TRY(stage(&dz2, z2, h->n, 2)); ST_TRY(stage(&dy2, y2, h->n, 3));
    EpiParams ep = base_epi(h);
    launch_state_out(h, ep, slot, dz1, dy1, dz2, dy2, st);
    if (g.p[0]) CU_TRY(h, cudaMemcpyAsync(z1, dz1, (size_t)h->N * 4, cudaMemcpyDeviceToHost, st));
    if (g.p[1]) CU_TRY(h, cudaMemcpyAsync(y1, dy1, (size_t)h->N * 4, cudaMemcpyDeviceToHost, st));
    if (g.p[2]) CU_TRY(h, cudaMemcpyAsync(z2, dz2, (size_t)h->n * 8, cudaMemcpyDeviceToHost, st));
    if (g.p[3]) CU_TRY(h, cudaMemcpyAsync(y2, dy2, (size_t)h->n * 8, cudaMemcpyDeviceToHost, st));
    CU_TRY(h, cudaStreamSynchronize(st));
    return ADMM_OK;
}

admm_status admm_get_preconditioner(admm_handle* h, double* D, double* R, double* Sinv) {
    if (!h) return ADMM_EINVAL;
    if (h->opt.dose_only) { h->err = "dose_only handle: no preconditioner"; return ADMM_ESTATE; }
    CU_TRY(h, cudaSetDevice(h->opt.device));
    if (D) for (int64_t i = 0; i < h->N; ++i) D[i] = 1.0 / (double)h->class_count[h->h_point_class[i]];
    if (R) memcpy(R, h->h_R.data(), (size_t)h->n * 8);
    if (Sinv) CU_TRY(h, cudaMemcpy2D(Sinv, (size_t)h->n * 8, h->d_Sinv, (size_t)h->lds * 8, (size_t)h->n * 8, (size_t)h->n, cudaMemcpyDeviceToHost));
    return ADMM_OK;
}

admm_status admm_get_timing(admm_handle* h, double ms[8], int64_t* plan_iters) {
    if (!h) return ADMM_EINVAL;
    if (ms) memcpy(ms, h->ms, sizeof h->ms);
    if (plan_iters) *plan_iters = h->plan_iters;
    return ADMM_OK;
}

admm_status admm_get_kernel_times(admm_handle* h, double total_ms[4], int64_t launches[4]) {
    if (!h) return ADMM_EINVAL;
    for (int k = 0; k < 4; ++k) {
        if (total_ms) total_ms[k] = h->ktimes.total_ms[k];
        if (launches) launches[k] = h->ktimes.launches[k];
    }
    return ADMM_OK;
}

}  // extern "C"
