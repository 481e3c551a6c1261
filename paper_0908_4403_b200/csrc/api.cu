// api.cu -- the extern "C" boundary of libheget.so (include/heget.h).  Argument checking,
// context bookkeeping and launches only; all arithmetic is in the kernels.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

#include "heget_internal.cuh"

namespace {

int fail_cuda(heget_ctx* ctx, cudaError_t err)
{
    if (ctx) snprintf(ctx->cuda_msg, sizeof(ctx->cuda_msg), "%s: %s", cudaGetErrorName(err), cudaGetErrorString(err));
    return HEGET_ECUDA;
}

struct DeviceGuard {
    int prev = -1;
    bool ok;
    explicit DeviceGuard(int dev)
    {
        ok = cudaGetDevice(&prev) == cudaSuccess && (prev == dev || cudaSetDevice(dev) == cudaSuccess);
        if (prev == dev) prev = -1;
    }
    ~DeviceGuard()
    {
        if (prev >= 0) cudaSetDevice(prev);
    }
};

void free_staging(heget_ctx* ctx)
{
    cudaFree(ctx->d_stage_mom);
    cudaFree(ctx->d_stage_w);
    cudaFree(ctx->d_stage_amp2);
    ctx->d_stage_mom = ctx->d_stage_w = ctx->d_stage_amp2 = nullptr;
    ctx->stage_events = ctx->stage_n_events = 0;
}

}  // namespace

namespace {
int gen_events(heget_ctx* ctx, uint64_t seed, int n, const heget_gen_cfg* cfg, uint64_t first_event, int64_t N,
               double* momenta, double* weight, void* stream)
{
    if (!ctx || !cfg || n < 2 || n > 8 || N < 0 || N > HEGET_MAX_EVENTS || (N > 0 && !momenta)) return HEGET_EINVAL;
    if (cfg->mode < HEGET_GEN_FIXED || cfg->mode > HEGET_GEN_TOYPDF || !(cfg->a > 0.0) || !std::isfinite(cfg->a)) return HEGET_EINVAL;
    if (cfg->mode == HEGET_GEN_LOGUNIFORM && (!(cfg->b >= cfg->a) || !std::isfinite(cfg->b) || !std::isfinite(cfg->y_max))) return HEGET_EINVAL;
    if (cfg->mode == HEGET_GEN_TOYPDF) {
        // tau = x1 x2 is drawn log-uniform in [tau_min, 1], tau_min = (n pt_cut)^2 / s (R19)
        const double tau_min = (n * ctx->pt_cut) * (n * ctx->pt_cut) / (cfg->a * cfg->a);
        if (!(tau_min > 0.0) || !(tau_min < 1.0)) return HEGET_EINVAL;
    }
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return fail_cuda(ctx, cudaGetLastError());
    int launches = 0;
    cudaError_t err = heget_launch_gen(ctx, seed, n, cfg, first_event, N, momenta, weight, (cudaStream_t)stream, &launches);
    ctx->launches += launches;
    return err == cudaSuccess ? HEGET_OK : fail_cuda(ctx, err);
}
}  // namespace

extern "C" {

int heget_init(int device, double alpha, double q_charge, double pt_cut, double eta_cut, double dr_cut,
               heget_ctx** out)
{
    if (!out || !(alpha > 0.0) || device < 0) return HEGET_EINVAL;
    if (!std::isfinite(alpha) || !std::isfinite(q_charge) || !std::isfinite(pt_cut) || !std::isfinite(eta_cut) ||
        !std::isfinite(dr_cut) || pt_cut < 0.0 || eta_cut < 0.0 || dr_cut < 0.0)
        return HEGET_EINVAL;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || device >= count) return HEGET_ECUDA;
    DeviceGuard guard(device);
    if (!guard.ok) return HEGET_ECUDA;
    heget_ctx* ctx = new (std::nothrow) heget_ctx();
    if (!ctx) return HEGET_ENOMEM;
    memset(ctx, 0, sizeof(*ctx));
    ctx->device = device;
    ctx->alpha = alpha;
    ctx->q_charge = q_charge;
    ctx->g = -q_charge * sqrt(4.0 * 3.14159265358979323846 * alpha);  // eq. (26)
    ctx->pt_cut = pt_cut;
    ctx->eta_cut = eta_cut;
    ctx->dr_cut = dr_cut;
    cudaDeviceProp prop;
    cudaError_t err = cudaGetDeviceProperties(&prop, device);
    if (err == cudaSuccess) {
        ctx->sm_count = prop.multiProcessorCount;
        err = cudaMalloc(&ctx->d_partials, sizeof(double) * 3 * kReduceBlocks * (HEGET_REDUCE_SLOTS + 1));
    }
    if (err == cudaSuccess) err = cudaMalloc(&ctx->d_stage_out3, sizeof(double) * 3);
    if (err == cudaSuccess) err = cudaStreamCreateWithFlags(&ctx->host_stream, cudaStreamNonBlocking);
    if (err == cudaSuccess) err = cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking);
    for (int c = 0; c < kHostChunks && err == cudaSuccess; ++c)
        err = cudaEventCreateWithFlags(&ctx->chunk_ready[c], cudaEventDisableTiming);
    if (err != cudaSuccess) {
        for (int c = 0; c < kHostChunks; ++c)
            if (ctx->chunk_ready[c]) cudaEventDestroy(ctx->chunk_ready[c]);
        if (ctx->host_stream) cudaStreamDestroy(ctx->host_stream);
        if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
        cudaFree(ctx->d_partials);
        cudaFree(ctx->d_stage_out3);
        delete ctx;
        return HEGET_ECUDA;
    }
    *out = ctx;
    return HEGET_OK;
}

void heget_destroy(heget_ctx* ctx)
{
    if (!ctx) return;
    DeviceGuard guard(ctx->device);
    free_staging(ctx);
    cudaFree(ctx->d_partials);
    cudaFree(ctx->d_stage_out3);
    for (int c = 0; c < kHostChunks; ++c)
        if (ctx->chunk_ready[c]) cudaEventDestroy(ctx->chunk_ready[c]);
    if (ctx->host_stream) cudaStreamDestroy(ctx->host_stream);
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    delete ctx;
}

const char* heget_strerror(int code)
{
    switch (code) {
        case HEGET_OK: return "success";
        case HEGET_EINVAL: return "invalid argument (n outside [2,8], N < 0 || N > HEGET_MAX_EVENTS, null pointer, bad precision or mode)";
        case HEGET_ECUDA: return "CUDA runtime error (see heget_last_cuda_error)";
        case HEGET_ENOMEM: return "allocation failed";
        case HEGET_ETOOBIG: return "batch larger than the fixed scratch of a no-allocation entry point (N > HEGET_NOALLOC_MAX_EVENTS)";
        default: return "unknown heget error code";
    }
}

const char* heget_last_cuda_error(const heget_ctx* ctx) { return ctx ? ctx->cuda_msg : ""; }

int64_t heget_launch_count(const heget_ctx* ctx) { return ctx ? ctx->launches : 0; }

int heget_gen_events(heget_ctx* ctx, uint64_t seed, int n, const heget_gen_cfg* cfg, uint64_t first_event,
                     int64_t N, double* momenta, double* weight, void* stream)
{
    if (N > 0 && !weight) return HEGET_EINVAL;   // only heget_rambo runs without a weight buffer
    if ((reinterpret_cast<uintptr_t>(momenta) & 15u) != 0) return HEGET_EINVAL;
    return gen_events(ctx, seed, n, cfg, first_event, N, momenta, weight, stream);
}

int heget_rambo(heget_ctx* ctx, uint64_t seed, int n, double sqrt_s_hat, int64_t N, double* momenta, void* stream)
{
    heget_gen_cfg cfg;
    cfg.mode = HEGET_GEN_FIXED;
    cfg.apply_cuts = 0;
    cfg.a = sqrt_s_hat;
    cfg.b = 0.0;
    cfg.y_max = 0.0;
    if ((reinterpret_cast<uintptr_t>(momenta) & 15u) != 0) return HEGET_EINVAL;
    return gen_events(ctx, seed, n, &cfg, 0, N, momenta, nullptr, stream);
}

int heget_amp2(heget_ctx* ctx, const double* momenta, int n, int precision, double* out_amp2, int64_t N, void* stream)
{
    return heget_amp2_algo(ctx, momenta, n, precision, HEGET_ALGO_TREE, out_amp2, N, stream);
}

int heget_amp2_algo(heget_ctx* ctx, const double* momenta, int n, int precision, int algo, double* out_amp2,
                    int64_t N, void* stream)
{
    if (algo < HEGET_ALGO_TREE || algo > HEGET_ALGO_TREE2) return HEGET_EINVAL;
    if (!ctx || n < 2 || n > 8 || N < 0 || N > HEGET_MAX_EVENTS || (N > 0 && (!momenta || !out_amp2))) return HEGET_EINVAL;
    if (precision != HEGET_FP32 && precision != HEGET_FP64) return HEGET_EINVAL;
    if ((reinterpret_cast<uintptr_t>(momenta) & 15u) != 0) return HEGET_EINVAL;
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return fail_cuda(ctx, cudaGetLastError());
    int launches = 0;
    cudaError_t err;
    if (algo == HEGET_ALGO_SUBSET)
        err = heget_launch_amp2_subset(ctx, momenta, n, precision, out_amp2, N, (cudaStream_t)stream, &launches);
    else if (algo == HEGET_ALGO_TREE2)
        err = heget_launch_amp2_twosided(ctx, momenta, n, precision, out_amp2, N, (cudaStream_t)stream, &launches);
    else
        err = heget_launch_amp2(ctx, momenta, n, precision, out_amp2, N, (cudaStream_t)stream, &launches);
    ctx->launches += launches;
    return err == cudaSuccess ? HEGET_OK : fail_cuda(ctx, err);
}

int heget_amp2_sampled(heget_ctx* ctx, uint64_t seed, uint64_t first_event, const double* momenta, int n,
                       int precision, double* out_amp2, int32_t* out_hel, int64_t N, void* stream)
{
    if (!ctx || n < 2 || n > 8 || N < 0 || N > HEGET_MAX_EVENTS || (N > 0 && (!momenta || !out_amp2))) return HEGET_EINVAL;
    if (precision != HEGET_FP32 && precision != HEGET_FP64) return HEGET_EINVAL;
    if ((reinterpret_cast<uintptr_t>(momenta) & 15u) != 0) return HEGET_EINVAL;
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return fail_cuda(ctx, cudaGetLastError());
    int launches = 0;
    cudaError_t err = heget_launch_amp2_sampled(ctx, seed, first_event, momenta, n, precision, out_amp2, out_hel, N,
                                                (cudaStream_t)stream, &launches);
    ctx->launches += launches;
    return err == cudaSuccess ? HEGET_OK : fail_cuda(ctx, err);
}

int heget_list2(heget_ctx* ctx, uint64_t seed, uint64_t first_event, const double* momenta, int n, int precision,
                double* out_amp2, int32_t* out_hel, int64_t N, void* stream)
{
    if (!ctx || n < 2 || n > 8 || N < 0 || N > HEGET_MAX_EVENTS || (N > 0 && (!momenta || !out_amp2))) return HEGET_EINVAL;
    if (precision != HEGET_FP32 && precision != HEGET_FP64) return HEGET_EINVAL;
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return fail_cuda(ctx, cudaGetLastError());
    int launches = 0;
    cudaError_t err = heget_launch_list2(ctx, seed, first_event, momenta, n, precision, out_amp2, out_hel, N, false,
                                         (cudaStream_t)stream, &launches);
    ctx->launches += launches;
    return err == cudaSuccess ? HEGET_OK : fail_cuda(ctx, err);
}

int heget_list2_sum(heget_ctx* ctx, const double* momenta, int n, int precision, double* out_amp2, int64_t N,
                    void* stream)
{
    if (!ctx || n < 2 || n > 8 || N < 0 || N > HEGET_MAX_EVENTS || (N > 0 && (!momenta || !out_amp2))) return HEGET_EINVAL;
    if (precision != HEGET_FP32 && precision != HEGET_FP64) return HEGET_EINVAL;
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return fail_cuda(ctx, cudaGetLastError());
    int launches = 0;
    cudaError_t err = heget_launch_list2(ctx, 0, 0, momenta, n, precision, out_amp2, nullptr, N, true,
                                         (cudaStream_t)stream, &launches);
    ctx->launches += launches;
    return err == cudaSuccess ? HEGET_OK : fail_cuda(ctx, err);
}

int heget_histogram(heget_ctx* ctx, const double* momenta, const double* value, int n, int64_t N, int observable,
                    double lo, double hi, int nbins, double* hist, void* stream)
{
    if (!ctx || n < 2 || n > 8 || N < 0 || N > HEGET_MAX_EVENTS || !hist || (N > 0 && (!momenta || !value))) return HEGET_EINVAL;
    if (observable < HEGET_OBS_PT_MAX || observable > HEGET_OBS_DR_ALL) return HEGET_EINVAL;
    if (nbins < 1 || nbins > HEGET_HIST_MAX_BINS || !(hi > lo)) return HEGET_EINVAL;
    if ((reinterpret_cast<uintptr_t>(momenta) & 15u) != 0) return HEGET_EINVAL;
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return fail_cuda(ctx, cudaGetLastError());
    int launches = 0;
    cudaError_t err = heget_launch_histogram(ctx, momenta, value, n, N, observable, lo, hi, nbins, hist,
                                             (cudaStream_t)stream, &launches);
    ctx->launches += launches;
    return err == cudaSuccess ? HEGET_OK : fail_cuda(ctx, err);
}

int heget_helas_wavefunction(heget_ctx* ctx, int fn, int precision, const double* p, int nhel, int ns, double* w,
                               int64_t N, void* stream)
{
    if (!ctx || N < 0 || N > HEGET_MAX_EVENTS || (N > 0 && (!p || !w))) return HEGET_EINVAL;
    if (fn < HEGET_FN_IXXXX0 || fn > HEGET_FN_VXXXX2) return HEGET_EINVAL;
    if (precision != HEGET_FP32 && precision != HEGET_FP64) return HEGET_EINVAL;
    if ((nhel != 1 && nhel != -1) || (ns != 1 && ns != -1)) return HEGET_EINVAL;
    if (((reinterpret_cast<uintptr_t>(p) | reinterpret_cast<uintptr_t>(w)) & 15u) != 0) return HEGET_EINVAL;
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return fail_cuda(ctx, cudaGetLastError());
    int launches = 0;
    cudaError_t err = heget_launch_helas_wavefunction(fn, precision, p, nhel, ns, w, N, (cudaStream_t)stream, &launches);
    ctx->launches += launches;
    return err == cudaSuccess ? HEGET_OK : fail_cuda(ctx, err);
}

int heget_helas_vertex(heget_ctx* ctx, int fn, int precision, const double* fi, const double* fo, const double* vc,
                       double g, double* out, int64_t N, void* stream)
{
    if (!ctx || N < 0 || N > HEGET_MAX_EVENTS || (N > 0 && !out)) return HEGET_EINVAL;
    if (fn < HEGET_VTX_IOVXXX || fn > HEGET_VTX_JIOXX0) return HEGET_EINVAL;
    if (precision != HEGET_FP32 && precision != HEGET_FP64) return HEGET_EINVAL;
    const bool need_fi = fn != HEGET_VTX_FVOXX0, need_fo = fn != HEGET_VTX_FVIXX0, need_vc = fn != HEGET_VTX_JIOXX0;
    if (N > 0 && ((need_fi && !fi) || (need_fo && !fo) || (need_vc && !vc))) return HEGET_EINVAL;
    if (((reinterpret_cast<uintptr_t>(fi) | reinterpret_cast<uintptr_t>(fo) | reinterpret_cast<uintptr_t>(vc) |
          reinterpret_cast<uintptr_t>(out)) & 15u) != 0)
        return HEGET_EINVAL;
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return fail_cuda(ctx, cudaGetLastError());
    int launches = 0;
    cudaError_t err = heget_launch_helas_vertex(fn, precision, fi, fo, vc, g, out, N, (cudaStream_t)stream, &launches);
    ctx->launches += launches;
    return err == cudaSuccess ? HEGET_OK : fail_cuda(ctx, err);
}

int heget_xsec_reduce(heget_ctx* ctx, const double* amp2, const double* weight, int n, int64_t N, double* out3,
                      void* stream)
{
    if (!ctx || n < 2 || n > 8 || N < 0 || N > HEGET_MAX_EVENTS || !out3 || (N > 0 && (!amp2 || !weight))) return HEGET_EINVAL;
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return fail_cuda(ctx, cudaGetLastError());
    int launches = 0;
    double* partials = ctx->d_partials + (size_t)(ctx->reduce_slot++ % HEGET_REDUCE_SLOTS) * 3 * kReduceBlocks;
    cudaError_t err = heget_launch_reduce(partials, amp2, weight, n, N, out3, (cudaStream_t)stream, &launches);
    ctx->launches += launches;
    return err == cudaSuccess ? HEGET_OK : fail_cuda(ctx, err);
}

int heget_xsec_reduce_noalloc(heget_ctx* ctx, const double* amp2, const double* weight, int n, int64_t N, double* out3,
                              void* stream)
{
    if (!ctx || n < 2 || n > 8 || N < 0 || !out3 || (N > 0 && (!amp2 || !weight))) return HEGET_EINVAL;
    if (N > HEGET_NOALLOC_MAX_EVENTS) {
        snprintf(ctx->cuda_msg, sizeof(ctx->cuda_msg), "heget_xsec_reduce_noalloc: N = %lld exceeds HEGET_NOALLOC_MAX_EVENTS = %lld",
                 (long long)N, (long long)HEGET_NOALLOC_MAX_EVENTS);
        return HEGET_ETOOBIG;
    }
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return fail_cuda(ctx, cudaGetLastError());
    int launches = 0;
    cudaError_t err = heget_launch_reduce_noalloc(ctx->device, amp2, weight, n, N, out3, (cudaStream_t)stream, &launches);
    ctx->launches += launches;
    return err == cudaSuccess ? HEGET_OK : fail_cuda(ctx, err);
}

int heget_xsec_host(heget_ctx* ctx, const double* momenta, const double* weight, int n, int precision, int64_t N,
                    double* out_amp2, double* out3)
{
    if (!ctx || n < 2 || n > 8 || N < 0 || N > HEGET_MAX_EVENTS || !out3 || (N > 0 && (!momenta || !weight))) return HEGET_EINVAL;
    if (precision != HEGET_FP32 && precision != HEGET_FP64) return HEGET_EINVAL;
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return fail_cuda(ctx, cudaGetLastError());
    const int64_t need = N * (n + 2);
    cudaError_t err = cudaSuccess;
    if (need > ctx->stage_events || N > ctx->stage_n_events) {
        free_staging(ctx);
        const int64_t cap_n = N > 0 ? N : 1;
        err = cudaMalloc(&ctx->d_stage_mom, sizeof(double) * 4 * cap_n * 10);
        if (err == cudaSuccess) err = cudaMalloc(&ctx->d_stage_w, sizeof(double) * cap_n);
        if (err == cudaSuccess) err = cudaMalloc(&ctx->d_stage_amp2, sizeof(double) * cap_n);
        if (err != cudaSuccess) {
            free_staging(ctx);
            snprintf(ctx->cuda_msg, sizeof(ctx->cuda_msg), "%s", cudaGetErrorString(err));
            return HEGET_ENOMEM;
        }
        ctx->stage_events = cap_n * 10;
        ctx->stage_n_events = cap_n;
    }
    cudaStream_t st = ctx->host_stream, cp = ctx->copy_stream;
    int launches = 0, l2 = 0;
    if (N > 0) {
        // H2D of chunk c+1 overlaps the amplitude kernel of chunk c (two streams, one event
        // per chunk); per-event results do not depend on how a batch is cut into launches
        const int chunks = (N >= 64 * 1024) ? kHostChunks : 1;
        const int64_t per = (N + chunks - 1) / chunks;
        const size_t ev_bytes = sizeof(double) * 4 * (size_t)(n + 2);
        err = cudaMemcpyAsync(ctx->d_stage_w, weight, sizeof(double) * N, cudaMemcpyHostToDevice, cp);
        for (int c = 0; c < chunks && err == cudaSuccess; ++c) {
            const int64_t lo = c * per, cnt = (lo + per <= N) ? per : N - lo;
            if (cnt <= 0) break;
            err = cudaMemcpyAsync(ctx->d_stage_mom + lo * 4 * (n + 2), momenta + lo * 4 * (n + 2), ev_bytes * cnt,
                                  cudaMemcpyHostToDevice, cp);
            if (err == cudaSuccess) err = cudaEventRecord(ctx->chunk_ready[c], cp);
            if (err == cudaSuccess) err = cudaStreamWaitEvent(st, ctx->chunk_ready[c], 0);
            int l1 = 0;
            if (err == cudaSuccess)
                err = heget_launch_amp2(ctx, ctx->d_stage_mom + lo * 4 * (n + 2), n, precision,
                                        ctx->d_stage_amp2 + lo, cnt, st, &l1);
            launches += l1;
        }
    }
    if (err == cudaSuccess)
        err = heget_launch_reduce(ctx->d_partials + (size_t)HEGET_REDUCE_SLOTS * 3 * kReduceBlocks, ctx->d_stage_amp2,
                                  ctx->d_stage_w, n, N, ctx->d_stage_out3, st, &l2);
    ctx->launches += launches + l2;
    if (err == cudaSuccess && out_amp2 && N > 0)
        err = cudaMemcpyAsync(out_amp2, ctx->d_stage_amp2, sizeof(double) * N, cudaMemcpyDeviceToHost, st);
    if (err == cudaSuccess) err = cudaMemcpyAsync(out3, ctx->d_stage_out3, sizeof(double) * 3, cudaMemcpyDeviceToHost, st);
    if (err == cudaSuccess) err = cudaStreamSynchronize(st);
    return err == cudaSuccess ? HEGET_OK : fail_cuda(ctx, err);
}

int heget_fma_peak(heget_ctx* ctx, int precision, double* flops_per_s)
{
    return heget_fma_peak_pattern(ctx, precision, HEGET_PEAK_CONST_OPERAND, flops_per_s);
}

int heget_fma_peak_pattern(heget_ctx* ctx, int precision, int pattern, double* flops_per_s)
{
    if (!ctx || !flops_per_s || (precision != HEGET_FP32 && precision != HEGET_FP64)) return HEGET_EINVAL;
    if (pattern < HEGET_PEAK_CONST_OPERAND || pattern > HEGET_PEAK_NODE_PATTERN) return HEGET_EINVAL;
    DeviceGuard guard(ctx->device);
    if (!guard.ok) return fail_cuda(ctx, cudaGetLastError());
    int launches = 0;
    cudaError_t err = heget_run_fma_peak(ctx, precision, pattern, flops_per_s, &launches);
    ctx->launches += launches;
    return err == cudaSuccess ? HEGET_OK : fail_cuda(ctx, err);
}

}  // extern "C"
