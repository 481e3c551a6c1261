// heget_internal.cuh -- shared declarations of libheget.so's translation units (product code).
// Nothing here is used by, or shared with, oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/heget.h"
#include "../../include/heget_bench.h"

constexpr int kHostChunks = 8;  // pipeline depth of heget_xsec_host

struct heget_ctx {
    int device;
    int sm_count;
    double alpha, q_charge;
    double g;  // gal[0] = gal[1] = -e Q_q (eq. 26)
    double pt_cut, eta_cut, dr_cut;
    // scratch owned by the context
    double* d_partials;     // [HEGET_REDUCE_SLOTS + 1][kReduceBlocks][3] block partial sums of heget_xsec_reduce:
                            // a ring used round-robin by the [dev] calls (they may run concurrently on
                            // different streams), the last slot is heget_xsec_host's own
    unsigned reduce_slot;   // next ring slot
    double* d_stage_mom;    // staging for the *_host entry point
    double* d_stage_w;
    double* d_stage_amp2;
    double* d_stage_out3;
    int64_t stage_events;   // capacity of the staging buffers, in events * (n+2)
    int64_t stage_n_events;
    cudaStream_t host_stream;   // compute stream of the *_host entry point
    cudaStream_t copy_stream;   // its H2D stream: chunk c+1 is copied while chunk c is computed
    cudaEvent_t chunk_ready[kHostChunks];
    int64_t launches;
    char cuda_msg[256];
};

constexpr int kReduceBlocks = 296;  // 2 CTAs per SM on a 148-SM B200; any value is correct

// launchers (each returns a cudaError_t from the launch)
cudaError_t heget_launch_amp2(const heget_ctx* ctx, const double* momenta, int n, int precision,
                              double* out_amp2, int64_t N, cudaStream_t stream, int* launches);
cudaError_t heget_launch_amp2_thread(const heget_ctx* ctx, const double* momenta, int n, int precision,
                                     double* out_amp2, int64_t N, cudaStream_t stream, int* launches);
cudaError_t heget_launch_amp2_subset(const heget_ctx* ctx, const double* momenta, int n, int precision,
                                     double* out_amp2, int64_t N, cudaStream_t stream, int* launches);
cudaError_t heget_launch_amp2_twosided(const heget_ctx* ctx, const double* momenta, int n, int precision,
                                       double* out_amp2, int64_t N, cudaStream_t stream, int* launches);
cudaError_t heget_launch_amp2_sampled(const heget_ctx* ctx, uint64_t seed, uint64_t first_event,
                                      const double* momenta, int n, int precision, double* out_amp2,
                                      int32_t* out_hel, int64_t N, cudaStream_t stream, int* launches);
cudaError_t heget_launch_list2(const heget_ctx* ctx, uint64_t seed, uint64_t first_event, const double* momenta,
                               int n, int precision, double* out_amp2, int32_t* out_hel, int64_t N, bool sum,
                               cudaStream_t stream, int* launches);
cudaError_t heget_launch_histogram(const heget_ctx* ctx, const double* momenta, const double* value, int n,
                                   int64_t N, int observable, double lo, double hi, int nbins, double* hist,
                                   cudaStream_t stream, int* launches);
cudaError_t heget_launch_helas_wavefunction(int fn, int precision, const double* p, int nhel, int ns, double* out,
                                            int64_t N, cudaStream_t stream, int* launches);
cudaError_t heget_launch_helas_vertex(int fn, int precision, const double* a, const double* b, const double* c,
                                      double g, double* out, int64_t N, cudaStream_t stream, int* launches);
cudaError_t heget_launch_gen(const heget_ctx* ctx, uint64_t seed, int n, const heget_gen_cfg* cfg,
                             uint64_t first_event, int64_t N, double* momenta, double* weight,
                             cudaStream_t stream, int* launches);
cudaError_t heget_launch_reduce(double* partials /* [kReduceBlocks][3] */, const double* amp2, const double* weight,
                                int n, int64_t N, double* out3, cudaStream_t stream, int* launches);
cudaError_t heget_launch_reduce_noalloc(int device /* current */, const double* amp2, const double* weight, int n, int64_t N,
                                        double* out3, cudaStream_t stream, int* launches);
cudaError_t heget_run_fma_peak(const heget_ctx* ctx, int precision, int pattern, double* flops_per_s, int* launches);
