// tables.cu -- tables built once per context: the stored angular-edge coefficients of the stage kernel (Eq.16-17, Eq.25),
// the upwind sign tables (Eq.24, Eq.25; parity helpers) and the signal-speed bound (R9).
#include <math.h>

#include "stage_math.cuh"

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

// ------------------------------------------------------------------------------------------------
// stored edge coefficients: q[cell][j][n] = s * dlambda_e * (c_e * n_0e) for the edge e that angle n owns in slot
// j (s = +1 if n is the edge's lower angle, else -1, so that q I_up is the flux LEAVING n), lowest mantissa bit
// = 1 if n is the upwind end.  c_e by the pinned 30-term chain (the one RAD_TAB_EDGE_SIGN reports).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_build_ke(const DeviceTables t, double *__restrict__ ke) {
    const long long nint = (long long)t.n[0] * t.n[1] * t.n[2];
    const long long total = nint * 3 * t.N;
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
        const int n = (int)(idx % t.N);
        const int jj = (int)((idx / t.N) % 3);
        const long long cint = idx / (3 * t.N);
        const int i = (int)(cint % t.n[0]) + t.ng, j = (int)((cint / t.n[0]) % t.n[1]) + t.ng, k = (int)(cint / ((long long)t.n[0] * t.n[1])) + t.ng;
        const long long c = ((long long)k * t.NJ + j) * t.NI + i;
        const int e = t.own_edge[n * 3 + jj];
        double q = 0.0;
        if (e >= 0) {
            const double *S = t.cell + c * RAD_NCELL + 5, *T = t.edge_T + (long long)e * 30;
            double acc = 0.0;
#pragma unroll
            for (int m = 0; m < 30; m++) acc = fma(S[m], T[m], acc);  // pinned 30-term chain
            const double ce = -acc;
            const double *cg = t.cell + c * RAD_NCELL;
            const double n0e = chain4(cg[1], cg[2], cg[3], cg[4], t.edge_mid[3 * e], t.edge_mid[3 * e + 1], t.edge_mid[3 * e + 2]);
            const bool owner_is_lo = t.edge_lo[e] == n;
            if (ce != 0.0) {
                q = (owner_is_lo ? t.edge_len[e] : -t.edge_len[e]) * (ce * n0e);
                const bool owner_up = (ce > 0.0) == owner_is_lo;
                long long bits = __double_as_longlong(q);
                bits = (bits & ~1ll) | (owner_up ? 1ll : 0ll);
                q = __longlong_as_double(bits);
            }
        }
        ke[idx] = q;
    }
}

}  // namespace

int launch_build_ke(const DeviceTables &t, double *ke, cudaStream_t s) {
    k_build_ke<<<t.sms * 8, 256, 0, s>>>(t, ke);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

int launch_sign_tables(const DeviceTables &t, signed char *face_sign, signed char *edge_sign, cudaStream_t s) {
    int launches = 0;
    if (face_sign) { k_face_signs<<<t.sms * 8, 256, 0, s>>>(t, face_sign); launches++; }
    if (edge_sign) { k_edge_signs<<<t.sms * 8, 256, 0, s>>>(t, edge_sign); launches++; }
    return cudaGetLastError() == cudaSuccess ? launches : -1;
}

int launch_maxspeed(const DeviceTables &t, double *out3, cudaStream_t s) {
    if (cudaMemsetAsync(out3, 0, 3 * sizeof(double), s) != cudaSuccess) return -1;
    k_maxspeed<<<t.sms * 4, 128, 0, s>>>(t, out3);
    return cudaGetLastError() == cudaSuccess ? 1 : -1;
}

}  // namespace rad
