// helas_eval.cu -- heget_helas_wavefunction / heget_helas_vertex: batched evaluation of the HEGET
// device functions of helas.cuh, one thread per element (product code).
// Buffers are fp64 in both precisions (as everywhere in this library); `precision` selects the
// arithmetic the functions run in.  A wavefunction is double[6][2] = cmplx w[6]
// (PAPER.md:553-554).
#include "helas.cuh"
#include "heget_internal.cuh"

namespace {

template <typename T>
__device__ __forceinline__ void load_w(const double* __restrict__ src, cmplx<T>* w)
{
    const double2* s = reinterpret_cast<const double2*>(src);
#pragma unroll
    for (int a = 0; a < 6; ++a) {
        const double2 v = s[a];
        w[a] = mkcmplx((T)v.x, (T)v.y);
    }
}

template <typename T>
__device__ __forceinline__ void store_w(const cmplx<T>* w, double* __restrict__ dst)
{
    double2* d = reinterpret_cast<double2*>(dst);
#pragma unroll
    for (int a = 0; a < 6; ++a) d[a] = make_double2((double)w[a].re, (double)w[a].im);
}

template <typename T>
__global__ void __launch_bounds__(256)
helas_wavefunction_kernel(int fn, const double* __restrict__ p, int nhel, int ns, double* __restrict__ out,
                          int64_t n)
{
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    const double2 a = reinterpret_cast<const double2*>(p)[2 * e], b = reinterpret_cast<const double2*>(p)[2 * e + 1];
    const T q[4] = {(T)a.x, (T)a.y, (T)b.x, (T)b.y};
    cmplx<T> w[6];
    switch (fn) {  // uniform over the launch
        case HEGET_FN_IXXXX0: ixxxx0(q, nhel, ns, w); break;
        case HEGET_FN_IXXXX1: ixxxx1(q, nhel, ns, w); break;
        case HEGET_FN_IXXXX2: ixxxx2(q, nhel, ns, w); break;
        case HEGET_FN_OXXXX0: oxxxx0(q, nhel, ns, w); break;
        case HEGET_FN_OXXXX1: oxxxx1(q, nhel, ns, w); break;
        case HEGET_FN_OXXXX2: oxxxx2(q, nhel, ns, w); break;
        case HEGET_FN_VXXXX0: vxxxx0(q, nhel, ns, w); break;
        case HEGET_FN_VXXXX1: vxxxx1(q, nhel, ns, w); break;
        default: vxxxx2(q, nhel, ns, w); break;
    }
    store_w(w, out + e * 12);
}

template <typename T>
__global__ void __launch_bounds__(256)
helas_vertex_kernel(int fn, const double* __restrict__ a, const double* __restrict__ b, const double* __restrict__ c,
                    double g, double* __restrict__ out, int64_t n)
{
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    cmplx<T> x[6], y[6], w[6];
    if (fn == HEGET_VTX_IOVXXX) {
        cmplx<T> z[6];
        load_w(a + e * 12, x);
        load_w(b + e * 12, y);
        load_w(c + e * 12, z);
        const cmplx<T> amp = iovxxx(x, y, z, (T)g);
        reinterpret_cast<double2*>(out)[e] = make_double2((double)amp.re, (double)amp.im);
        return;
    }
    if (fn == HEGET_VTX_FVIXX0) {
        load_w(a + e * 12, x);
        load_w(c + e * 12, y);
        fvixx0(x, y, (T)g, w);
    } else if (fn == HEGET_VTX_FVOXX0) {
        load_w(b + e * 12, x);
        load_w(c + e * 12, y);
        fvoxx0(x, y, (T)g, w);
    } else {
        load_w(a + e * 12, x);
        load_w(b + e * 12, y);
        jioxx0(x, y, (T)g, w);
    }
    store_w(w, out + e * 12);
}

}  // namespace

cudaError_t heget_launch_helas_wavefunction(int fn, int precision, const double* p, int nhel, int ns, double* out,
                                            int64_t N, cudaStream_t stream, int* launches)
{
    *launches = 0;
    if (N == 0) return cudaSuccess;
    *launches = 1;
    const unsigned blocks = (unsigned)((N + 255) / 256);
    if (precision == HEGET_FP32)
        helas_wavefunction_kernel<float><<<blocks, 256, 0, stream>>>(fn, p, nhel, ns, out, N);
    else
        helas_wavefunction_kernel<double><<<blocks, 256, 0, stream>>>(fn, p, nhel, ns, out, N);
    return cudaGetLastError();
}

cudaError_t heget_launch_helas_vertex(int fn, int precision, const double* a, const double* b, const double* c,
                                      double g, double* out, int64_t N, cudaStream_t stream, int* launches)
{
    *launches = 0;
    if (N == 0) return cudaSuccess;
    *launches = 1;
    const unsigned blocks = (unsigned)((N + 255) / 256);
    if (precision == HEGET_FP32)
        helas_vertex_kernel<float><<<blocks, 256, 0, stream>>>(fn, a, b, c, g, out, N);
    else
        helas_vertex_kernel<double><<<blocks, 256, 0, stream>>>(fn, a, b, c, g, out, N);
    return cudaGetLastError();
}
