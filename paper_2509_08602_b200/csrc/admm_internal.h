// Internal declarations shared by the translation units of libadmm_b200.so.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/admm_b200.h"

constexpr int kMaxClasses = 8;
constexpr int kTileM = 128;        // rows of the big (Phi-side) operand per UMMA tile
constexpr int kBlockK = 32;        // fp32 elements per k-block = one 128-byte swizzle row
constexpr int kBoxRows = 32;       // rows per TMA box of the big operand (partial tiles load fewer boxes)
constexpr int kMaxBpad = 512;      // slots in the per-plan tables / partial-sum arrays (B <= 512)
constexpr int kMaxMmaN = 256;      // plans per contraction pass (UMMA N limit); larger batches run in chunks
constexpr double kRhoFloorDiv = 65536.0;   // default rho rule: w_BOT is clamped below at w0 / kRhoFloorDiv (reading R8)
constexpr int kNumResid = 5;       // ||x-z+||^2, ||z+-z||^2, ||x||^2, ||z+||^2, ||y+||^2

// One unit of work of a contraction kernel: a 128-row tile of the big operand times a k-range.
struct TcUnit {
    int32_t row0;      // first row of the tile in the big operand
    int32_t rows;      // valid rows (1..128)
    int32_t kb0;       // first k-block (of 32 elements)
    int32_t kb_count;  // number of k-blocks (>= 1)
    int32_t slot;      // K1: partial-sum slot this unit writes
    int32_t pad;
};

// Epilogue selector of the contraction kernels
enum { EPI_K1_PARTIAL = 0, EPI_K3_STATE = 1, EPI_OBJECTIVE = 2, EPI_RAW = 3 };

// Everything the epilogues need.  Plan-major ("slot-major") layouts: a plan's vector is contiguous.
struct EpiParams {
    // common
    int32_t slot0;              // first slot of this contraction pass (chunk of <= 256 plans)
    int32_t n_slots_active;     // live slots of this pass: slot0 .. slot0 + n_slots_active - 1 (the HOST's upper bound)
    const int32_t* bact_dev;    // device scalar: live slots of the whole batch right now (nullptr: n_slots_active is exact).
                                // The host's bound lags the device by up to one check interval; see eff_nact().
    int32_t n_mma;              // UMMA N (multiple of 16, >= n_slots_active)
    int64_t N, n;               // points, time variables
    int64_t ldN, ldn;           // row strides of [slot][N] and [slot][n] arrays (elements)
    // K1: partial[slot][plan][128] fp32
    float* partial;
    // K3 / objective
    const uint8_t* point_class;     // [N]
    const uint32_t* mask;           // [B][mask_words] or nullptr
    const int32_t* slot_plan;       // [Bpad] plan index of each slot (mask row)
    int64_t mask_words;
    const float* utab;              // [kMaxClasses][kMaxBpad] u_hat per (class, slot)
    const float* crtab;             // [kMaxClasses][kMaxBpad] c_hat / rho per (class, slot)
    float a_cls[kMaxClasses];       // sigma_k * D_k
    float sense[kMaxClasses];
    float thr[kMaxClasses];
    float* s1;                      // [Bpad][ldN] single state s = x + y of block 1
    void* g_hi;                     // [Bpad][ldN] operand of K1: head of a (2 z1 - s1 - c/rho): fp32 on the tf32 grid, or bf16
    void* g_lo;                     // [Bpad][ldN] tail
    int32_t small_bf16;             // 1: the small operands (G, V, T) are emitted as bf16 hi/lo pairs (ADMM_STORAGE_BF16)
    float* resid_partial;           // [grid][kMaxBpad][kNumResid] per-CTA residual sums (nullptr: not this iteration)
    double* hinge_partial;          // objective: [grid][kMaxBpad][kMaxClasses]
    float* qraw;                    // EPI_RAW (test hook): raw accumulators [slot][ldN]
};

// Live slots of this pass as the DEVICE knows them: the compaction kernel shrinks *bact_dev, the host's n_slots_active (which
// sized the launch: n_mma, grids) follows one check interval later.
__host__ __device__ inline int eff_nact(const EpiParams& ep) {
#ifdef __CUDA_ARCH__
    if (ep.bact_dev) {
        const int live = *ep.bact_dev - ep.slot0;
        return live < 0 ? 0 : (live < ep.n_slots_active ? live : ep.n_slots_active);
    }
#endif
    return ep.n_slots_active;
}

struct TcLaunch {
    CUtensorMap map_big;     // big operand, tile-major [tiles * 128][32], box {32, 32}
    CUtensorMap map_big128;  // same tensor, box {32, 128}: a whole 16 KB tile per TMA (fp32 path)
    int32_t big_kb_total;    // k-blocks per row tile of the big operand (tile (rt, kb) starts at row (rt * big_kb_total + kb) * 128)
    CUtensorMap map_small_hi;// small operand [Bpad][K], box {32, n_mma}
    CUtensorMap map_small_lo;
    const TcUnit* units;     // device
    const int32_t* cta_unit_begin;  // device [grid + 1]
    int32_t grid;
    int32_t mma_passes;      // 3: 3xTF32 with on-chip split of the big operand; 2: big operand already on the tf32 grid
    int32_t epi;
    int32_t kblk;            // elements per k-block = per 128-byte row: 32 (fp32 / tf32) or 64 (bf16)
    int32_t mma_kind;        // 0: kind::tf32, 1: kind::f16 with bf16 operands
    int32_t n_sa, n_sb;      // fp32 kernel: depth of the big / small operand rings in shared memory
    int32_t chunk_kb;        // > 0: drain the TMEM accumulator every chunk_kb k-blocks (fp32 path, n_mma <= 128); 0: never
    float debias;            // drained sums are multiplied by (1 + debias): the accumulator's truncation, put back on average
    EpiParams ep;
};

struct KernelTimes {
    double total_ms[4] = {0, 0, 0, 0};
    int64_t launches[4] = {0, 0, 0, 0};
};

struct admm_handle {
    admm_options opt{};
    cudaStream_t stream = nullptr;
    int sm_count = 148;
    int64_t N = 0, n = 0, ldN = 0, ldn = 0;
    int n_classes = 0;
    admm_class classes[kMaxClasses]{};
    int64_t class_count[kMaxClasses]{};
    std::vector<uint8_t> h_point_class;

    // device, owned
    float* d_phi = nullptr;        // [N][ldn] row-major (setup; kept only by the SIMT cross-check path)
    float* d_phiT = nullptr;       // [n][ldN] row-major (SIMT cross-check path only)
    float* d_phi_t = nullptr;      // tile-major Phi:   [ceil(N/128)][ceil(n/32)][128][32]  (K3 / objective big operand)
    float* d_phiT_t = nullptr;     // tile-major Phi^T: [ceil(n/128)][ceil(N/32)][128][32]  (K1 big operand)
    // ADMM_STORAGE_CSR: thresholded Phi as CSR (rows = points) and the CSR of Phi^T (rows = time variables)
    int64_t *d_csr_ptr = nullptr, *d_csrT_ptr = nullptr; int32_t *d_csr_col = nullptr, *d_csrT_col = nullptr;
    float *d_csr_val = nullptr, *d_csrT_val = nullptr; int64_t csr_nnz = 0; float csr_tau = 0.f;
    float* d_small_t = nullptr;    // [max(N, n)][<= 256] element-major copy of the plan operand of one SpMM
    uint8_t* d_point_class = nullptr;
    double* d_R = nullptr;         // [n]
    double* d_Rb = nullptr;        // [n] R o bot_rows: b_hat = d_Rb * w_BOT (Eq. 13: only the isocenter rows carry w_BOT with the coupling blocks)
    double* d_bot = nullptr;       // [n] bot_rows as 0.0 / 1.0
    double* d_Sinv = nullptr;      // [n][lds], lds = n rounded up to even (16-byte rows for cp.async), pad = 0
    int64_t lds = 0;
    int kblk = 32;                 // elements per 128-byte k-block of the stored Phi: 32 (fp32) or 64 (bf16 storage)
    int k2_rows = 16;              // rows of the K2b block tile: 16 / 32 / 40 / 48 / 64 (k2_choose_rows, when the batch buffers are allocated)
    std::vector<double> h_R;

    // per-solve state (reallocated when B grows)
    int32_t B = 0, Bpad = 0;
    float *d_s1 = nullptr, *d_ghi = nullptr, *d_glo = nullptr;        // [Bpad][ldN]; d_glo = d_ghi + Bpad * ldN (one allocation: planes of a 3-D tensor map)
    double* d_s2 = nullptr;                                           // [Bpad][ldn]
    double* d_rhs = nullptr;                                          // [Bpad][ldn]
    float *d_vhi = nullptr, *d_vlo = nullptr;                         // [Bpad][ldn]; d_vlo = d_vhi + Bpad * ldn (same)
    float* d_partial = nullptr; int64_t partial_slots = 0;            // [slots][Bpad][128]
    float* d_resid1 = nullptr;                                        // [grid][kMaxBpad][5]
    double* d_resid2 = nullptr;                                       // [blocks][kMaxBpad][5]
    double* d_hinge = nullptr;                                        // [grid][kMaxBpad][kMaxClasses]
    uint32_t* d_mask = nullptr; int64_t mask_words = 0; bool has_mask = false; int64_t mask_capacity = 0;
    int32_t* d_slot_plan = nullptr;
    float *d_utab = nullptr, *d_crtab = nullptr;
    double *d_beta = nullptr, *d_rho = nullptr;                       // per slot
    int32_t* d_active_counts = nullptr;                               // [B][kMaxClasses]
    int32_t* d_conv_flags = nullptr;                                  // [Bpad] stopping-rule / presolve verdict per slot
    int32_t* d_bact = nullptr;                                        // device scalar: live slots (H5 shrinks it on the device)
    int32_t* d_moves = nullptr; int32_t* d_nmoves = nullptr;          // compaction: [Bpad/2][2] slot pairs + their count
    int32_t* d_iters_plan = nullptr; float* d_res_plan = nullptr;     // per PLAN: iterations done, residual norms [B][2]
    double* d_wnorm = nullptr;                                        // [kMaxBpad][kMaxClasses] w_k / N_kp per slot
    float* d_t_f32 = nullptr; double* d_obj = nullptr;                // finalise: t [Bpad][ldn], objective per slot
    int32_t* d_plan_slot = nullptr; float* d_tout = nullptr;          // outputs in plan order
    float* d_qbuf = nullptr;                                          // SIMT / CSR path: Q [pass][ldN]
    int32_t* h_bact_ring = nullptr;                                   // pinned host ring the live count is copied into after every check
    cudaEvent_t bact_ev[8] = {};                                      // one event per ring entry
    int k2_attr_tj = 0;                                               // block tile of the K2b instantiation whose smem opt-in is set
    struct MapKey { int kind, slot0, n_mma; CUtensorMap big, big128, hi, lo; };
    std::vector<MapKey> map_cache;                                    // tensor maps per (contraction, slot0, n_mma); cleared on reallocation
    TcUnit* d_units_k1 = nullptr; int32_t* d_cta_begin_k1 = nullptr; int grid_k1 = 0; int slots_k1 = 0;
    int32_t* d_mtile_slot_begin = nullptr;                            // [m_tiles + 1]
    TcUnit* d_units_k3 = nullptr; int32_t* d_cta_begin_k3 = nullptr; int grid_k3 = 0;
    std::vector<int32_t> slot_plan, plan_slot, iters;
    bool solved = false;
    int32_t presolved = 0;                                            // plans of the last solve settled by the presolve

    double ms[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    int64_t plan_iters = 0;
    int64_t launch_count = 0;
    KernelTimes ktimes;
    std::string err;
};

// ---- gemm_tc.cu
admm_status tc_init(admm_handle* h);                       // resolves cuTensorMapEncodeTiled, sets smem attribute
admm_status tc_make_map(admm_handle* h, CUtensorMap* out, const void* base, int64_t rows, int64_t cols,
                        int64_t ld_elems, int box_rows, int elem_bytes = 4);
admm_status tc_launch(admm_handle* h, const TcLaunch& L);

// ---- csr.cu
admm_status csr_threshold(admm_handle* h);
admm_status csr_build(admm_handle* h);
void launch_csr_k1(admm_handle* h, int slot0, int nact, int n_mma, cudaStream_t s);
void launch_csr_k3(admm_handle* h, int nact, const float* vhi, const float* vlo, float* qbuf, cudaStream_t s);

// ---- kernels.cu  (everything that is not a tcgen05 contraction)
void launch_pack_tiles(const float* src, int64_t src_rows, int64_t src_cols, int64_t ld_src, bool transpose, float* dst, cudaStream_t s);
void launch_pack_tiles_bf16(const float* src, int64_t src_rows, int64_t src_cols, int64_t ld_src, bool transpose, void* dst, cudaStream_t s);
void launch_round_bf16(float* x, int64_t count, cudaStream_t s);
void launch_transpose(const float* src, int64_t rows, int64_t cols, int64_t ld_src, float* dst, int64_t ld_dst, cudaStream_t s);
void launch_scale_rows_to_f64(const float* phi, int64_t ld, int64_t row0, int64_t rows, int64_t n,
                              const uint8_t* cls, const double* a_cls, double* out, cudaStream_t s);
void launch_round_tf32(float* x, int64_t count, cudaStream_t s);
void launch_finish_S(double* M, int64_t n, double* R, cudaStream_t s);      // M -> S = I + R M R (in place), R from diag
void launch_symmetrize(double* A, int64_t n, cudaStream_t s);
void launch_count_active(const uint32_t* mask, int64_t mask_words, const uint8_t* cls, int64_t N, int B,
                         int32_t* counts, cudaStream_t s);
void launch_emit_g(const EpiParams& ep, int Bact, cudaStream_t s);          // G from the current s1 (start / warm start)
void launch_k2a(admm_handle* h, int slot0, int nact, int n_mma, cudaStream_t s);
void launch_k2b(admm_handle* h, int Bact, bool resid, cudaStream_t s);
void launch_simt_k1(admm_handle* h, int slot0, int nact, int n_mma, int splits, cudaStream_t s);
void launch_simt_k3(admm_handle* h, const EpiParams& ep, int epi, const float* vhi, const float* vlo, float* qbuf, cudaStream_t s);
void launch_convergence(admm_handle* h, int Bact, int grid1, int grid2, float tol, float eps_abs, int it, cudaStream_t s);
void launch_compaction(admm_handle* h, int Bact, cudaStream_t s);
void launch_presolve_state(const EpiParams& ep, int B, cudaStream_t s);
void launch_presolve_test(admm_handle* h, int slot0, int nact, int n_mma, double margin, cudaStream_t s);
void launch_presolve_reset(admm_handle* h, int B, cudaStream_t s);
void launch_init_plan_records(admm_handle* h, int B, cudaStream_t s);
void launch_make_t(admm_handle* h, int Bact, void* t_hi, void* t_lo, float* t_f32, cudaStream_t s);
void launch_objective_reduce(admm_handle* h, int B, int grid, const float* t_f32, const double* wnorm, double* obj_slot, cudaStream_t s);
void launch_lowdose_volume(const float* dose, int64_t ld, int64_t N, int B, float lo, float hi, uint32_t* in_vol, int64_t words,
                           uint32_t* any_vol, cudaStream_t s);
void launch_gather_rows(const float* src, int64_t ld, const int32_t* plan_slot, int B, int64_t n, float* dst, cudaStream_t s);
void launch_state_out(admm_handle* h, const EpiParams& ep, int slot, float* z1, float* y1, double* z2, double* y2, cudaStream_t s);
int k2b_grid(const admm_handle* h, int Bact);
int k2_choose_rows(const admm_handle* h, int Bpad);
void launch_split_small(const float* x, int64_t count, int64_t ld, void* hi, void* lo, bool bf16, cudaStream_t s);
void launch_reduce_partial(admm_handle* h, int nact, int n_mma, double* out, cudaStream_t s);
