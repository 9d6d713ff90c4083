// image.cuh -- image (a7), offset gather (a8), layout conversion and sampling kernels.
#pragma once
#include "common.cuh"

namespace rtm {

// a7 (Eq. 3): I[x] (+)= scale * sum_k Uz[k][x] Vz[k][x].  Thread = one physical z-quad.
__global__ void __launch_bounds__(256) image_kernel(Layout L, const float *__restrict__ U, const float *__restrict__ V,
                                                    int r, float scale, int accumulate, float *__restrict__ img) {
    const int nq = L.upz / 4;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long rows = (long long)L.nx * L.ny;
    if (t >= rows * nq) return;
    const long long row = t / nq;
    const int iz = (int)(t % nq) * 4;
    if (iz >= L.nz) return;
    const long long o = row * L.upz + iz;
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 4
    for (int k = 0; k < r; k++) {
        const float4 u = ldcs4(U + k * L.Nu + o), v = ldcs4(V + k * L.Nu + o);
        acc.x = fmaf(u.x, v.x, acc.x);
        acc.y = fmaf(u.y, v.y, acc.y);
        acc.z = fmaf(u.z, v.z, acc.z);
        acc.w = fmaf(u.w, v.w, acc.w);
    }
    const float res[4] = {acc.x, acc.y, acc.z, acc.w};
    float *out = img + row * L.nz + iz;
    for (int q = 0; q < 4 && iz + q < L.nz; q++) out[q] = accumulate ? fmaf(scale, res[q], out[q]) : scale * res[q];
}

// a8 (Eq. 4): G[ih][x] = scale * sum_k Uz[k][x + h e_x] Vz[k][x - h e_x].
// Thread = one physical z-quad of one row, loops over offsets and probes.  rest = ny * upz / 4 quads
// per x (x is the slowest axis, so a shift by h is a shift by h * ny * upz floats).
__global__ void __launch_bounds__(256) gather_kernel(Layout L, const float *__restrict__ U, const float *__restrict__ V,
                                                     int r, int nh, const int *__restrict__ offs, float scale,
                                                     float *__restrict__ G) {
    const int nq = L.upz / 4;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long rows = (long long)L.nx * L.ny;
    if (t >= rows * nq) return;
    const long long row = t / nq;
    const int iz = (int)(t % nq) * 4;
    if (iz >= L.nz) return;
    const int ix = (int)(row / L.ny);
    const long long xs = (long long)L.ny * L.upz;
    const long long o = row * L.upz + iz;
    const long long N = rows * L.nz;
    for (int ih = 0; ih < nh; ih++) {
        const int h = offs[ih];
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        if (ix + h >= 0 && ix + h < L.nx && ix - h >= 0 && ix - h < L.nx) {
            const float *pu = U + o + h * xs, *pv = V + o - h * xs;
#pragma unroll 4
            for (int k = 0; k < r; k++) {
                const float4 u = ld4(pu + k * L.Nu), v = ld4(pv + k * L.Nu);
                acc.x = fmaf(u.x, v.x, acc.x);
                acc.y = fmaf(u.y, v.y, acc.y);
                acc.z = fmaf(u.z, v.z, acc.z);
                acc.w = fmaf(u.w, v.w, acc.w);
            }
        }
        const float res[4] = {acc.x, acc.y, acc.z, acc.w};
        float *out = G + (long long)ih * N + row * L.nz + iz;
        for (int q = 0; q < 4 && iz + q < L.nz; q++) out[q] = scale * res[q];
    }
}

// canonical [Np] -> internal haloed/pitched layout (halo untouched: it is zeroed once at create)
__global__ void pack_field_kernel(Layout L, const float *__restrict__ src, float *__restrict__ dst) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long Np = (long long)L.Px * L.Py * L.Pz;
    if (t >= Np) return;
    const int jz = (int)(t % L.Pz);
    const long long q = t / L.Pz;
    const int jy = (int)(q % L.Py), jx = (int)(q / L.Py);
    dst[L.org + jx * L.sx + jy * L.sy + jz] = src[t];
}
__global__ void unpack_field_kernel(Layout L, const float *__restrict__ src, float *__restrict__ dst) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long Np = (long long)L.Px * L.Py * L.Pz;
    if (t >= Np) return;
    const int jz = (int)(t % L.Pz);
    const long long q = t / L.Pz;
    const int jy = (int)(q % L.Py), jx = (int)(q / L.Py);
    dst[t] = src[L.org + jx * L.sx + jy * L.sy + jz];
}
// internal probe planes -> canonical [r][N]
__global__ void unpack_probes_kernel(Layout L, int r, const float *__restrict__ src, float *__restrict__ dst) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long N = (long long)L.nx * L.ny * L.nz;
    if (t >= N * r) return;
    const int k = (int)(t / N);
    const long long x = t % N;
    const int iz = (int)(x % L.nz);
    const long long row = x / L.nz;
    dst[t] = src[k * L.Nu + row * L.upz + iz];
}
// Z [nt][r] -> internal [nt][zr] (zr = r rounded up to 8, zero padded) so that rows are float4-aligned
__global__ void pack_probes_kernel(int nt, int r, int zr, const float *__restrict__ src, float *__restrict__ dst) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (long long)nt * zr) return;
    const int k = (int)(t % zr);
    const long long n = t / zr;
    dst[t] = k < r ? src[n * r + k] : 0.0f;
}
// per-axis K1 table: k1[j] = (1 - s_j) / (1 + s_j) (1 where s_j = 0), same arithmetic as k1_of in the step kernels
__global__ void k1_table_kernel(const float *__restrict__ damp, float *__restrict__ k1, int n) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) k1[i] = k1_of(damp[i]);
}
// stand-alone sampling of the current field (the last step of a pass has no following step kernel)
__global__ void __launch_bounds__(256) sample_kernel(const StepArgs a) { sample_points(a, blockIdx.x, 256, threadIdx.x); }

}  // namespace rtm

namespace rtm {

// Time-blocked probe accumulation (a5/a6 with T steps per flush):
//   PZ[k][x] += sum_{j < ncur} Z[n_j][k] * hist[j][x],   n_j = n_0 + j*dir  (dir = +1 forward, -1 adjoint)
// Same sums as T per-step rank-1 updates, applied in step order j = 0..ncur-1 per (k, x), so the result does
// not depend on T's grouping beyond fp32 rounding of the partial sums.  Thread = one physical z-quad; the T
// history quads stay in registers while the r probe planes stream through once (8 r N bytes per T steps).
template <int T>
__global__ void __launch_bounds__(256) probe_flush_kernel(Layout L, const float *__restrict__ hist, int ncur,
                                                          const float *__restrict__ Z0, long long zstep, int zr,
                                                          int r, float *__restrict__ PZ) {
    __shared__ __align__(16) float sz[T * 256];   // [T][zr], zr <= 256
    for (int i = threadIdx.x; i < T * zr; i += 256) {
        const int j = i / zr, k = i % zr;
        sz[i] = j < ncur ? Z0[j * zstep + k] : 0.0f;
    }
    __syncthreads();
    const int nq = L.upz / 4;
    const long long t = (long long)blockIdx.x * 256 + threadIdx.x;
    const long long rows = (long long)L.nx * L.ny;
    if (t >= rows * nq) return;
    const long long row = t / nq;
    const int iz = (int)(t % nq) * 4;
    if (iz >= L.nz) return;
    const long long o = row * L.upz + iz;
    float4 h[T];
#pragma unroll
    for (int j = 0; j < T; j++) h[j] = j < ncur ? ld4(hist + j * L.Nu + o) : make_float4(0.f, 0.f, 0.f, 0.f);
    float *p = PZ + o;
    float4 nxt[4];
#pragma unroll
    for (int i = 0; i < 4; i++) nxt[i] = (i < r) ? ldcs4(p + (long long)i * L.Nu) : make_float4(0.f, 0.f, 0.f, 0.f);
    for (int k = 0; k < r; k += 4) {   // zr is a multiple of 8 and rows beyond r are zero-padded
        float4 acc[4];
#pragma unroll
        for (int i = 0; i < 4; i++) acc[i] = nxt[i];
#pragma unroll
        for (int i = 0; i < 4; i++)
            nxt[i] = (k + 4 + i < r) ? ldcs4(p + (long long)(k + 4 + i) * L.Nu) : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
        for (int j = 0; j < T; j++) {
            const float4 z = ld4(sz + j * zr + k);
            const float zz[4] = {z.x, z.y, z.z, z.w};
#pragma unroll
            for (int i = 0; i < 4; i++) {
                acc[i].x = fmaf(zz[i], h[j].x, acc[i].x);
                acc[i].y = fmaf(zz[i], h[j].y, acc[i].y);
                acc[i].z = fmaf(zz[i], h[j].z, acc[i].z);
                acc[i].w = fmaf(zz[i], h[j].w, acc[i].w);
            }
        }
#pragma unroll
        for (int i = 0; i < 4; i++)
            if (k + i < r) stcs4(p + (long long)(k + i) * L.Nu, acc[i]);
    }
}

}  // namespace rtm
