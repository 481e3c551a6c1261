// gen.cu -- heget_rambo / heget_gen_events: device-side Philox4x32-10 + RAMBO + boost + cuts +
// weight, one thread per event (product code; step 4 of PAPER.md:116-122, cuts of eq. 9
// PAPER.md:89-96, weight from eqs. 1-4).  The paper draws its random numbers
// on the CPU and copies them over; here the counter-based generator runs
// in the kernel, keyed by the global event index, so nothing crosses PCIe.
#include "heget_internal.cuh"
#include "philox.cuh"

namespace {

// key = seed, counter = (event_lo, event_hi, slot, 0); u = (x + 0.5) 2^-32 in (0,1)
__device__ __forceinline__ void uniforms4(uint64_t seed, uint64_t event, uint32_t slot, double u[4])
{
    uint32_t x[4];
    philox4x32_10((uint32_t)event, (uint32_t)(event >> 32), slot, 0u, (uint32_t)seed, (uint32_t)(seed >> 32), x);
#pragma unroll
    for (int i = 0; i < 4; ++i) u[i] = ((double)x[i] + 0.5) * (1.0 / 4294967296.0);
}

__device__ __forceinline__ double phase_space_volume(int n, double s)
{
    // Phi_n(s) = (2 pi)^(4-3n) (pi/2)^(n-1) s^(n-2) / ((n-1)! (n-2)!)   (integral of eq. 4)
    const double pi = 3.14159265358979323846;
    double v = 1.0 / (8.0 * pi);  // n = 2
    for (int m = 3; m <= n; ++m) v *= s * (pi / 2.0) / ((2.0 * pi) * (2.0 * pi) * (2.0 * pi)) / ((double)(m - 1) * (double)(m - 2));
    return v;
}

constexpr int kGenThreads = 128;

// One thread per event computes; the CTA's momenta go through shared memory (row stride padded by one
// 16-byte word: conflict-free stores) and leave as ONE contiguous span of double2 words, the mirror of
// MomentaTile::load in amp2_common.cuh (a thread writing its own (n+2) x 32 bytes at a stride of
// 32 (n+2) bytes reached 20 % of the HBM write rate).
template <int N>
__global__ void __launch_bounds__(kGenThreads)
gen_kernel(uint64_t seed, heget_gen_cfg cfg, double pt_cut, double eta_cut, double dr_cut,
           uint64_t first_event, int64_t n_events, double* __restrict__ momenta, double* __restrict__ weight)
{
    constexpr int WORDS = 2 * (N + 2);             // double2 words per event
    constexpr int STRIDE = WORDS + 1;
    __shared__ double2 s_out[kGenThreads * STRIDE];
    const int64_t ev0 = (int64_t)blockIdx.x * kGenThreads;
    int64_t e = ev0 + threadIdx.x;
    const bool live = e < n_events;
    if (!live) e = n_events - 1;                   // past the end: recompute the last event, store nothing
    const uint64_t ev = first_event + (uint64_t)e;
    const double pi = 3.14159265358979323846;

    double u0[4];
    uniforms4(seed, ev, 0u, u0);
    double rs, y, extra = 1.0;
    if (cfg.mode == HEGET_GEN_FIXED) {
        rs = cfg.a;
        y = 0.0;
    } else if (cfg.mode == HEGET_GEN_LOGUNIFORM) {
        rs = cfg.a * exp(u0[0] * log(cfg.b / cfg.a));   // a (b/a)^u; the logarithm is loop-invariant
        y = cfg.y_max * (2.0 * u0[1] - 1.0);
    } else {
        const double s = cfg.a * cfg.a;
        const double tau_min = (N * pt_cut) * (N * pt_cut) / s;
        const double ln_tau_min = log(tau_min);
        const double ln_tau = (1.0 - u0[0]) * ln_tau_min;
        const double tau = exp(ln_tau);
        y = (2.0 * u0[1] - 1.0) * (-0.5 * ln_tau);
        const double x1 = sqrt(tau) * exp(y), x2 = sqrt(tau) * exp(-y);
        const double o1 = 1.0 - x1, o2 = 1.0 - x2;
        const double f1 = o1 * o1 * o1 / sqrt(x1), f2 = o2 * o2 * o2 / sqrt(x2);
        rs = sqrt(tau * s);
        extra = tau * (-ln_tau_min) * (-ln_tau) * 2.0 * f1 * f2;
    }

    // RAMBO: isotropic massless q_i, then the conformal boost and rescale to total (rs, 0)
    double q[N][4], Q[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
    for (int i = 0; i < N; ++i) {
        double u[4];
        uniforms4(seed, ev, (uint32_t)(i + 1), u);
        const double c = 2.0 * u[0] - 1.0;
        const double s = sqrt(1.0 - c * c);
        double sf, cf;
        sincospi(2.0 * u[1], &sf, &cf);   // phi = 2 pi u: no range reduction needed
        const double q0 = -log(u[2] * u[3]);
        q[i][0] = q0; q[i][1] = q0 * s * cf; q[i][2] = q0 * s * sf; q[i][3] = q0 * c;
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) Q[mu] += q[i][mu];
    }
    const double M = sqrt(Q[0] * Q[0] - Q[1] * Q[1] - Q[2] * Q[2] - Q[3] * Q[3]);
    const double inv_m = 1.0 / M;   // one division instead of five
    const double b[3] = {-Q[1] * inv_m, -Q[2] * inv_m, -Q[3] * inv_m};
    const double gam = Q[0] * inv_m, a = 1.0 / (1.0 + gam), x = rs * inv_m;
    // boost by y along z from one exponential: cosh, sinh and the beam energies (the error of sinh y
    // from the difference is 1e-16 absolute, i.e. of k0 sinh y relative to the scale sqrt(s_hat))
    const double ey = exp(y), emy = 1.0 / ey;
    const double ch = 0.5 * (ey + emy), sh = 0.5 * (ey - emy);

    double2* out = s_out + threadIdx.x * STRIDE;
    const double e1 = 0.5 * rs * ey, e2 = 0.5 * rs * emy;
    out[0] = make_double2(e1, 0.0);
    out[1] = make_double2(0.0, e1);
    out[2] = make_double2(e2, 0.0);
    out[3] = make_double2(0.0, -e2);

    bool pass = true;
    double eta[N], phi[N];
#pragma unroll
    for (int i = 0; i < N; ++i) {
        const double bq = b[0] * q[i][1] + b[1] * q[i][2] + b[2] * q[i][3];
        const double k0 = x * (gam * q[i][0] + bq);
        const double kx = x * (q[i][1] + b[0] * q[i][0] + a * bq * b[0]);
        const double ky = x * (q[i][2] + b[1] * q[i][0] + a * bq * b[1]);
        const double kz = x * (q[i][3] + b[2] * q[i][0] + a * bq * b[2]);
        const double E = k0 * ch + kz * sh;   // boost by y along z
        const double pz = kz * ch + k0 * sh;
        out[4 + 2 * i] = make_double2(E, kx);
        out[5 + 2 * i] = make_double2(ky, pz);
        if (cfg.apply_cuts) {
            // massless: asinh(pz / pT) = sign(pz) log((E + |pz|) / pT), one logarithm and one reciprocal square root;
            // pT > pT_cut is taken on the squares
            const double pt2 = kx * kx + ky * ky;
            eta[i] = copysign(log((E + fabs(pz)) * rsqrt(pt2)), pz);
            phi[i] = atan2(ky, kx);
            pass = pass && (pt2 > pt_cut * pt_cut) && (fabs(eta[i]) < eta_cut);
        }
    }
    if (cfg.apply_cuts) {
#pragma unroll
        for (int i = 0; i < N; ++i)
#pragma unroll
            for (int j = i + 1; j < N; ++j) {
                const double deta = eta[i] - eta[j];
                double dphi = fabs(phi[i] - phi[j]);
                if (dphi > pi) dphi = 2.0 * pi - dphi;
                pass = pass && (deta * deta + dphi * dphi > dr_cut * dr_cut);
            }
    }
    if (weight && live) {
        const double shat = rs * rs;
        weight[e] = pass ? phase_space_volume(N, shat) / (2.0 * shat) * extra : 0.0;
    }
    __syncthreads();
    const int64_t left = n_events - ev0;
    const int span = (int)(left < kGenThreads ? left : kGenThreads) * WORDS;
    double2* dst = reinterpret_cast<double2*>(momenta) + ev0 * WORDS;
    for (int idx = threadIdx.x; idx < span; idx += kGenThreads) dst[idx] = s_out[(idx / WORDS) * STRIDE + idx % WORDS];
}

template <int N>
cudaError_t launch(const heget_ctx* ctx, uint64_t seed, const heget_gen_cfg& cfg, uint64_t first_event,
                   int64_t n_events, double* momenta, double* weight, cudaStream_t stream)
{
    const int threads = kGenThreads;
    const int64_t blocks = (n_events + threads - 1) / threads;
    gen_kernel<N><<<(unsigned)blocks, threads, 0, stream>>>(seed, cfg, ctx->pt_cut, ctx->eta_cut, ctx->dr_cut,
                                                           first_event, n_events, momenta, weight);
    return cudaGetLastError();
}

}  // namespace

cudaError_t heget_launch_gen(const heget_ctx* ctx, uint64_t seed, int n, const heget_gen_cfg* cfg,
                             uint64_t first_event, int64_t N, double* momenta, double* weight,
                             cudaStream_t stream, int* launches)
{
    *launches = 0;
    if (N == 0) return cudaSuccess;
    *launches = 1;
    switch (n) {
        case 2: return launch<2>(ctx, seed, *cfg, first_event, N, momenta, weight, stream);
        case 3: return launch<3>(ctx, seed, *cfg, first_event, N, momenta, weight, stream);
        case 4: return launch<4>(ctx, seed, *cfg, first_event, N, momenta, weight, stream);
        case 5: return launch<5>(ctx, seed, *cfg, first_event, N, momenta, weight, stream);
        case 6: return launch<6>(ctx, seed, *cfg, first_event, N, momenta, weight, stream);
        case 7: return launch<7>(ctx, seed, *cfg, first_event, N, momenta, weight, stream);
        case 8: return launch<8>(ctx, seed, *cfg, first_event, N, momenta, weight, stream);
        default: return cudaErrorInvalidValue;
    }
}
