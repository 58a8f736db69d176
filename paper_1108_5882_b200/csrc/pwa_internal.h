// pwa_internal.h — context and shared device helpers of libpwa.so (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/pwa.h"

namespace pwa {

constexpr int kMaxFastWaves = 64;     // V passed by value for n <= 64
constexpr int kMaxRes = 64;
constexpr int kMaxAng = 4;
constexpr int kMaxK = 1024;

// Result record of one evaluation k, written by the finishing block of the data pass:
//   [0] nll  [1] L_data  [2] Norm  [3] n_nonfinite  [4 + 2a] d nll/d Re V_a  [5 + 2a] d nll/d Im V_a
inline int result_stride(int n) { return 4 + 2 * n; }
// Partial / data-term component order: [0] L_data [1] n_nonfinite [2 + 2a] Re T_a [3 + 2a] Im T_a
inline int n_components(int n) { return 2 + 2 * n; }

struct VArg { double v[2 * kMaxFastWaves]; };   // kernel-parameter copy of V (<= 1 KB)

struct Sample {
    // constant-resonance form
    void *amps = nullptr;   bool amps_owned = false;
    // factored form
    double *mass = nullptr; void *ang = nullptr; bool fact_owned = false; int n_ang = 0;
    bool factored = false;
    double *weights = nullptr; bool weights_owned = false;   // optional per-event weights (NEXT-3), [n_events]
    double sum_w = 0.0;     // sum of the weights (compensated, index order; found once in pwa_set_weights): N_data of eq. 2
    int64_t n_events = -1;  // -1 = not uploaded
    int64_t n_gen = 0;
};

struct ResParams {           // by-value kernel argument in factored mode
    double m2[kMaxRes];      // M_r^2
    double mg[kMaxRes];      // M_r * G_r
};

}  // namespace pwa

struct pwa_ctx {
    int n = 0;
    pwa_dtype storage = PWA_F64;
    int device = 0;
    cudaStream_t stream = nullptr;
    int sm_count = 148;
    pwa::Sample data, mc;
    // floating mode
    int n_res = 0;
    cudaEvent_t ev_V = nullptr; bool ev_V_pending = false;   // recorded after the H2D copy of the staged V (h_V may be refilled only after it)
    std::vector<int32_t> res_of_wave, ang_of_wave;
    std::vector<int32_t> wave_of_pair;        // [n_res * kMaxAng] -> wave or -1
    std::vector<double> mass0, width0;
    bool res_set = false;
    // normalisation matrix
    double *d_M = nullptr;                    // [n][n][2]
    std::vector<double> h_M;
    bool M_valid = false;
    int M_path = 0;                           // 0 = FP64 build, 1 = int8 tcgen05 build (norm_i8.cu)
    // scratch
    double *d_partials = nullptr; size_t partials_cap = 0;   // doubles
    unsigned *d_ticket = nullptr;
    // result records [kMaxK][result_stride] live in device-mapped pinned HOST memory: the finishing block
    // writes them there and sets h_flags[k] = seq (no D2H copy, the host polls the flag)
    double *h_result = nullptr, *dev_result = nullptr;
    double *d_result = nullptr;                               // device scratch records (res_grad, microbench)
    unsigned long long *h_flags = nullptr, *dev_flags = nullptr;   // [kMaxK]
    unsigned long long seq = 0;                               // id of the most recent enqueue
    double *d_V = nullptr; double *h_V = nullptr;            // [kMaxK][n][2]
    double *d_scratch = nullptr; size_t scratch_cap = 0;     // bytes (M partials, batch partials)
    double *d_H = nullptr;                                    // [2n][2n] Fumili matrix (allocated on first use)
    int last_K = 0;
    int batch_path = -1;                                      // family of the most recent batched call (pwa_batch_path)
    // cached TMA descriptor of the DATA sample (data_term_tma.cu); rebuilt when the key changes
    struct { const void *base = nullptr; long long n_events = -1; int box_rows = 0; bool valid = false;
             alignas(64) unsigned char map[128]; } tmap_cache;
    // int8 tensor-core M build (norm_i8.cu): per-column power-of-two scales found at MC upload
    struct { bool valid = false; int exp[128]; float scale[128]; double cmax[128]; } i8q;
    // int8 tensor-core batched evaluation (batch_i8.cu): the same for the DATA sample, found on first use
    struct { bool checked = false, valid = false; int exp[128]; float scale[128]; double cmax[128];
             unsigned char *planes = nullptr; } i8d;       // planes: X digit-plane image of the sample (k_bi8_planes), library-owned
    // resident evaluation grid (option "resident"; data_term_tma.cu): mailbox in device-mapped pinned host memory
    // ([0] = sequence number, [1 ..] = V) and its device copy
    unsigned long long *h_cmd = nullptr, *dev_cmd_host = nullptr, *d_cmd = nullptr;
    unsigned long long *h_rres = nullptr, *dev_rres = nullptr;      // tagged result record of the resident grid (mapped host memory)
    bool opt_resident = false, resident_running = false;
    uint64_t launches = 0;
    int opt_data_term = 0, opt_norm = 0, opt_batch = 0;
    int opt_l2_resident_mb = -1;              // MB of the data sample's head kept in L2 between evaluations (TMA data term); -1 = automatic, 0 = off
    int opt_likelihood = 0;                   // 0 = eq. 3 extended form (default), 1 = eq. 2 normalised form
    int opt_fix_phase = 0;                    // minimisers: 0 = all parameters free, k = gauge Im V_(k-1) = 0 (pwa_fix_phase_host)
    std::string err;
};

namespace pwa {

pwa_status fail(pwa_ctx *ctx, pwa_status s, const std::string &msg);
pwa_status cuda_fail(pwa_ctx *ctx, cudaError_t e, const char *what);
pwa_status ensure_partials(pwa_ctx *ctx, size_t doubles);
// N_data of the eq. 2 form: the number of data events, or the sum of their weights for a weighted sample
inline double eq2_n_data(const pwa_ctx *ctx) { return ctx->data.weights ? ctx->data.sum_w : (double)(ctx->data.n_events > 0 ? ctx->data.n_events : 0); }
pwa_status ensure_scratch(pwa_ctx *ctx, size_t bytes);

#define PWA_CUDA(ctx, call)                                                   \
    do {                                                                      \
        cudaError_t e__ = (call);                                             \
        if (e__ != cudaSuccess) return pwa::cuda_fail((ctx), e__, #call);     \
    } while (0)

// launchers (one .cu each)
pwa_status launch_data_term(pwa_ctx *ctx, const double *V_host_k, int k, double *out_dev_terms);
pwa_status launch_batch(pwa_ctx *ctx, int K);   // V already staged in h_V/d_V
pwa_status launch_norm_build(pwa_ctx *ctx);
pwa_status launch_fumili(pwa_ctx *ctx, double *H_dev, bool with_norm);   // norm_dmma.cu (row-scaled Gram over DATA)
pwa_status prepare_norm_i8(pwa_ctx *ctx);                  // norm_i8.cu: after a constant-resonance MC upload
pwa_status launch_norm_i8(pwa_ctx *ctx, bool *handled, bool three_planes);    // norm_i8.cu
double norm_i8_error_bound(const pwa_ctx *ctx);
pwa_status i8_column_scales(pwa_ctx *ctx, const void *amps, long long n_events, int D, int *exp, float *scale,
                            double *cmax, bool *valid);    // norm_i8.cu
pwa_status launch_batch_i8(pwa_ctx *ctx, int K, bool *handled);   // batch_i8.cu
double batch_i8_error_estimate(const pwa_ctx *ctx);               // batch_i8.cu
pwa_status launch_res_grad(pwa_ctx *ctx, const double *V, double *dM, double *dG);
pwa_status launch_resident(pwa_ctx *ctx, bool *started);   // data_term.cu
pwa_status launch_floating_passes(pwa_ctx *ctx, const double *V, int *ncomp_out);   // factored.cu
pwa_status run_microbench(pwa_ctx *ctx, int which, int64_t bytes, double *result);

}  // namespace pwa
