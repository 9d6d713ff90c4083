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

// a8 with vector offsets h = (hx, hy) on 3D grids (Eq. 4; reading C28):
//   G[ih][x] = scale * sum_k Uz[k][x + hx e_x + hy e_y] Vz[k][x - hx e_x - hy e_y], zero where a shifted point leaves
// [0,nx) x [0,ny).  trip = [nl][3] = (ih, hx, hy): the offsets the register-tiled kernel did not take.
__global__ void __launch_bounds__(256) gather_xy_kernel(Layout L, const float *__restrict__ U, const float *__restrict__ V,
                                                        int r, int nl, const int *__restrict__ trip, float scale,
                                                        float *__restrict__ G) {
    const int nq = L.upz / 4;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long rows = (long long)L.nx * L.ny;
    if (t >= rows * nq) return;
    const long long row = t / nq;
    const int iz = (int)(t % nq) * 4;
    if (iz >= L.nz) return;
    const int ix = (int)(row / L.ny), iy = (int)(row % L.ny);
    const long long xs = (long long)L.ny * L.upz;
    const long long o = row * L.upz + iz;
    const long long N = rows * L.nz;
    for (int i = 0; i < nl; i++) {
        const int ih = trip[3 * i], hx = trip[3 * i + 1], hy = trip[3 * i + 2];
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        if (ix + hx >= 0 && ix + hx < L.nx && ix - hx >= 0 && ix - hx < L.nx && iy + hy >= 0 && iy + hy < L.ny &&
            iy - hy >= 0 && iy - hy < L.ny) {
            const long long sh = hx * xs + (long long)hy * L.upz;
            const float *pu = U + o + sh, *pv = V + o - sh;
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

// a8, register-tiled fast path for a run of consecutive offsets h0, h0+1, ..., h0+nh-1 (nh <= GT_HP).
//
// The generic kernel above reads 2 x LDG.128 per 4 FMA and is bound by L1/L2 throughput (c3: 1.39 ms for a 552 MB
// minimum).  Here a block owns GT_X consecutive x and 32 consecutive floats of the fast axes (z, or (y,z) in 3D: a
// shift by h along x is a shift by whole rows of R = ny*upz floats) and all offsets; a thread owns an 8 (x) by 8 (h)
// patch of outputs of one lane.  Per probe k the block stages the GT_X + GT_HP - 1 rows of U and of V it needs in
// shared memory (cp.async, double-buffered, zero-filled outside [0, nx): Eq. 4's terms vanish there, reading C11);
// a thread then reads 15 + 15 values and does 64 FMAs: acc[i][j] += U[i + j] * V[i - j + 7].
// Same products in the same order (k ascending, one fma each) as the generic kernel and as image_kernel, so
// gather[h = 0] stays bit-identical to the image.
// HP = offsets per launch: 48 (c3's 41 offsets in one launch) or 16 (the short hx runs of (hx, hy) volumes: 47 instead
// of 79 staged rows per tile, 8 warps instead of 24).
constexpr int GT_X = 32, GT_HP = 48;
__host__ __device__ constexpr int gt_rows(int hp) { return GT_X + hp - 1; }
__host__ __device__ constexpr int gt_threads(int hp) { return 32 * (GT_X / 8) * (hp / 8); }
__host__ __device__ constexpr int gt_stages(int hp) { return 4; }   // probes in flight (shared-memory buffers)
__host__ __device__ constexpr int gt_smem(int hp) { return gt_stages(hp) * 2 * gt_rows(hp) * 32 * 4; }

template <int HP, bool XY>
__global__ void __launch_bounds__(gt_threads(HP)) gather_tiled_kernel(Layout L, const float *__restrict__ U,
                                                                   const float *__restrict__ V, int r, int nh, int h0,
                                                                   const int4 *__restrict__ runs, int nruns, float scale,
                                                                   float *__restrict__ G) {
    constexpr int GT_ROWS = gt_rows(HP), GT_THREADS = gt_threads(HP), NST = gt_stages(HP);
    extern __shared__ __align__(16) float gsm[];   // [NST buffers][U | V][GT_ROWS][32]
    const int tid = threadIdx.x, lane = tid & 31, grp = tid >> 5;
    const int xg = grp % (GT_X / 8), hg = grp / (GT_X / 8);
    const long long R = (long long)L.ny * L.upz;
    // 1-D offsets: grid (l blocks, x tiles), one run (nh, h0).  (hx, hy) volumes: ONE launch for all runs of this HP
    // class, runs[i] = (h0, hy, nh, first output plane); 1-D grid ordered (y row; run; z block; x tile fastest), so
    // that the blocks sharing halo rows in x run together, and so do the runs that read the same rows of Uz / Vz at
    // different hy (U row iy + hy of run hy is U row (iy + 1) + (hy - 1) of the next y row): the planes come from DRAM
    // about once per launch instead of once per run (c4, 9 x 3 offsets: 3 reads of 8.6 GB -> 1).
    int hy = 0;
    long long l0;
    int x0;
    if (XY) {
        const int nxt = (L.nx + GT_X - 1) / GT_X, nlz = L.upz / 32;
        unsigned b = blockIdx.x;
        x0 = (int)(b % nxt) * GT_X; b /= nxt;
        const int lz = (int)(b % nlz); b /= nlz;
        const int4 rn = runs[b % nruns];
        const int iy = (int)(b / nruns);
        h0 = rn.x; hy = rn.y; nh = rn.z;
        G += (long long)rn.w * L.nx * L.ny * L.nz;
        l0 = ((long long)iy * nlz + lz) * 32;
    } else {
        l0 = (long long)blockIdx.x * 32;          // first float of the fast axes
        x0 = blockIdx.y * GT_X;
    }
    const int xu0 = x0 + h0, xv0 = x0 - (h0 + HP - 1);     // first x row of the U / V tile
    // vector offsets (hx, hy) on 3D grids (reading C28): upz % 32 == 0, so the block's 32 floats lie in one y row
    // iy0 and a shift by hy along y is a shift by hy * upz floats, valid for the whole block or for none of it
    if (XY) {
        const int iy0 = (int)(l0 / L.upz);
        const bool yok = iy0 + hy >= 0 && iy0 + hy < L.ny && iy0 - hy >= 0 && iy0 - hy < L.ny;
        if (!yok) r = 0;                                       // every term vanishes (C28): the block writes zeros
        U += (long long)hy * L.upz;
        V -= (long long)hy * L.upz;
    }

    // Per-thread chunk table of the staging loop (16-offset instance): source pointer and shared-memory offset of each
    // of its 16-byte chunks are the same for every probe up to + k * Nu, so the row / bound / 64-bit address arithmetic
    // is done once, not r times (ncu, c4 xy volume: 289 warp instructions per probe and warp, 64 of them FMA).
    constexpr int NCH = (2 * GT_ROWS * 8 + GT_THREADS - 1) / GT_THREADS;
    const float *csrc[HP == 16 ? NCH : 1];
    int cdst[HP == 16 ? NCH : 1];
    if (HP == 16) {
#pragma unroll
        for (int i = 0; i < NCH; i++) {
            const int c = tid + i * GT_THREADS;
            const int row = c >> 3, q = c & 7;
            const bool isV = row >= GT_ROWS;
            const int x = isV ? xv0 + (row - GT_ROWS) : xu0 + row;
            const bool ok = c < 2 * GT_ROWS * 8 && x >= 0 && x < L.nx;
            csrc[i] = ok ? (isV ? V : U) + (long long)x * R + l0 + q * 4 : nullptr;
            cdst[i] = c < 2 * GT_ROWS * 8 ? row * 32 + q * 4 : -1;
        }
    }
    auto request = [&](int k, int buf) {
        float *dst = gsm + buf * (2 * GT_ROWS * 32);
        if (HP == 16) {
#pragma unroll
            for (int i = 0; i < NCH; i++)
                if (cdst[i] >= 0) cp_async16(dst + cdst[i], csrc[i] ? csrc[i] + (long long)k * L.Nu : U + l0, csrc[i] != nullptr);
            cp_async_commit();
            return;
        }
        // 2 * GT_ROWS rows of 128 bytes = 8 chunks of 16 bytes each
        for (int c = tid; c < 2 * GT_ROWS * 8; c += GT_THREADS) {
            const int row = c >> 3, q = c & 7;
            const bool isV = row >= GT_ROWS;
            const int x = isV ? xv0 + (row - GT_ROWS) : xu0 + row;
            const bool ok = x >= 0 && x < L.nx;
            const float *src = (isV ? V : U) + (long long)k * L.Nu + (long long)(ok ? x : 0) * R + l0 + q * 4;
            cp_async16(dst + row * 32 + q * 4, src, ok);
        }
        cp_async_commit();
    };

    float acc[8][8];
#pragma unroll
    for (int i = 0; i < 8; i++)
#pragma unroll
        for (int j = 0; j < 8; j++) acc[i][j] = 0.f;

    // NST - 1 probes in flight ahead of the one being consumed; one commit group per probe slot (empty past the end)
#pragma unroll
    for (int q = 0; q < NST - 1; q++) {
        if (q < r) request(q, q);
        else cp_async_commit();
    }
    for (int k = 0; k < r; k++) {
        cp_async_wait<NST - 2>();
        __syncthreads();            // probe k has landed for everybody; nobody still reads the buffer of probe k - 1
        if (k + NST - 1 < r) request(k + NST - 1, (k + NST - 1) % NST);
        else cp_async_commit();
        const float *us = gsm + (k % NST) * (2 * GT_ROWS * 32) + (8 * (xg + hg)) * 32 + lane;
        const float *vs = gsm + (k % NST) * (2 * GT_ROWS * 32) + (GT_ROWS + 8 * xg - 8 * hg + HP - 8) * 32 + lane;
        float u[15], v[15];
#pragma unroll
        for (int m = 0; m < 15; m++) { u[m] = us[m * 32]; v[m] = vs[m * 32]; }
#pragma unroll
        for (int i = 0; i < 8; i++)
#pragma unroll
            for (int j = 0; j < 8; j++) acc[i][j] = fmaf(u[i + j], v[i - j + 7], acc[i][j]);
    }

    // canonical output [nh][nx][ny][nz]: lane -> (iy, iz) of the pitch-padded fast axes
    const long long l = l0 + lane;
    const int iy = (int)(l / L.upz), iz = (int)(l - (long long)iy * L.upz);
    if (iz >= L.nz || iy >= L.ny) return;
    const long long N = (long long)L.nx * L.ny * L.nz;
#pragma unroll
    for (int i = 0; i < 8; i++) {
        const int x = x0 + xg * 8 + i;
        if (x >= L.nx) break;
#pragma unroll
        for (int j = 0; j < 8; j++) {
            const int ih = hg * 8 + j;
            if (ih < nh) G[(long long)ih * N + ((long long)x * L.ny + iy) * L.nz + iz] = scale * acc[i][j];
        }
    }
}

// canonical [Np] -> internal haloed/pitched layout (halo untouched: it is zeroed once at create)
__global__ void pack_field_kernel(Layout L, const float *__restrict__ src, float *__restrict__ dst) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long Np = (long long)L.Px * L.Py * L.Pzc;
    if (t >= Np) return;
    const int jz = (int)(t % L.Pzc);
    const long long q = t / L.Pzc;
    const int jy = (int)(q % L.Py), jx = (int)(q / L.Py);
    dst[L.org + jx * L.sx + jy * L.sy + jz + L.zs] = src[t];
}
__global__ void unpack_field_kernel(Layout L, const float *__restrict__ src, float *__restrict__ dst) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long Np = (long long)L.Px * L.Py * L.Pzc;
    if (t >= Np) return;
    const int jz = (int)(t % L.Pzc);
    const long long q = t / L.Pzc;
    const int jy = (int)(q % L.Py), jx = (int)(q / L.Py);
    dst[t] = src[L.org + jx * L.sx + jy * L.sy + jz + L.zs];
}
// internal probe planes -> canonical [r][N]
// two != 0 (probe_fields = 2): r counts all 2 r_probes planes; canonical plane f r_probes + k = internal plane 2k + f
__global__ void unpack_probes_kernel(Layout L, int r, int two, const float *__restrict__ src, float *__restrict__ dst) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long N = (long long)L.nx * L.ny * L.nz;
    if (t >= N * r) return;
    int k = (int)(t / N);
    if (two) { const int rh = r / 2; k = k < rh ? 2 * k : 2 * (k - rh) + 1; }
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
    __shared__ __align__(16) float sz[(T <= 16 ? T : 16) * 256];   // [T][zr]; zr <= 256 (T <= 16), zr <= 128 (T = 32)
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
