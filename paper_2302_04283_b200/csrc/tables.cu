// tables.cu -- parity helpers: the upwind sign tables (Eq.24, Eq.25) and the signal-speed bound (R9).
#include <math.h>

#include "rad_internal.h"

namespace rad {
namespace {

__device__ __forceinline__ signed char sgn(double x) { return (signed char)((x > 0.0) - (x < 0.0)); }

__global__ void k_face_signs(DeviceTables t, signed char *__restrict__ out) {
    const long long total = t.ncell * 3 * t.N;
    for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < total; q += (long long)gridDim.x * blockDim.x) {
        const int n = (int)(q % t.N);
        const long long cf = q / t.N;  // cell*3 + axis
        const double *f = t.face + cf * RAD_NFACE;
        const double na = fma(f[3], t.nhat[3 * n + 2], fma(f[2], t.nhat[3 * n + 1], fma(f[1], t.nhat[3 * n], f[0])));
        out[q] = sgn(na);
    }
}

__global__ void k_edge_signs(DeviceTables t, signed char *__restrict__ out) {
    const long long total = t.ncell * t.E;
    for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < total; q += (long long)gridDim.x * blockDim.x) {
        const int e = (int)(q % t.E);
        const double *S = t.cell + (q / t.E) * RAD_NCELL + 5, *T = t.edge_T + (long long)e * 30;
        double acc = 0.0;
        for (int w = 0; w < 30; w++) acc = fma(S[w], T[w], acc);
        out[q] = sgn(-acc);
    }
}

__global__ void k_maxspeed(DeviceTables t, double *__restrict__ out3) {
    // |n^a / n^0| at faces; n^0 at the face = -1/E_0hat.  One warp-reduced atomic max per block (values >= 0,
    // so the IEEE bit pattern orders like an unsigned integer).
    double mx[3] = {0.0, 0.0, 0.0};
    const long long total = t.ncell * 3;
    for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < total; q += (long long)gridDim.x * blockDim.x) {
        const double *f = t.face + q * RAD_NFACE;
        const int ax = (int)(q % 3);
        const double alpha_f = -f[4];
        double m = 0.0;
        for (int n = 0; n < t.N; n++) {
            const double na = fma(f[3], t.nhat[3 * n + 2], fma(f[2], t.nhat[3 * n + 1], fma(f[1], t.nhat[3 * n], f[0])));
            m = fmax(m, fabs(na * alpha_f));
        }
        mx[ax] = fmax(mx[ax], m);
    }
    for (int ax = 0; ax < 3; ax++) {
        double v = mx[ax];
        for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
        if ((threadIdx.x & 31) == 0) atomicMax(reinterpret_cast<unsigned long long *>(out3 + ax), (unsigned long long)__double_as_longlong(v));
    }
}

}  // namespace

int launch_sign_tables(const DeviceTables &t, signed char *face_sign, signed char *edge_sign, cudaStream_t s) {
    int launches = 0;
    if (face_sign) { k_face_signs<<<148 * 8, 256, 0, s>>>(t, face_sign); launches++; }
    if (edge_sign) { k_edge_signs<<<148 * 8, 256, 0, s>>>(t, edge_sign); launches++; }
    return cudaGetLastError() == cudaSuccess ? launches : -1;
}

int launch_maxspeed(const DeviceTables &t, double *out3, cudaStream_t s) {
    if (cudaMemsetAsync(out3, 0, 3 * sizeof(double), s) != cudaSuccess) return -1;
    k_maxspeed<<<148 * 4, 128, 0, s>>>(t, out3);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace rad
