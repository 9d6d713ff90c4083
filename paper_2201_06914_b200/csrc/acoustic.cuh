// acoustic.cuh -- isotropic acoustic time step (a1) with fused damping, source injection (a3),
// deferred receiver sampling (a4) and the probe accumulated in EVERY step (a5; schedule (A) of DESIGN.md,
// probe_block <= 1).  2D and 3D.  Time-blocked probing uses acoustic2d_stream.cuh / acoustic3d_stream.cuh.
//
//   du_new = K1 du + K2 * sum_axes sum_j w_j (u[+j] - 2u + u[-j])      (increment form of O2:
//   u_new  = u + du_new                                                 du = u_cur - u_prev)
//
// Thread = one z-quad (4 consecutive z, float4) of one (jx[,jy]) row.  Neighbours come straight from
// global memory: in 2D the fields (7 MB) are L2-resident and the block's 8 rows share L1; the probe
// planes are the only DRAM stream (byte model).
#pragma once
#include "common.cuh"

namespace rtm {

#define ACC_AXIS(P, M)                                  \
    {                                                   \
        s[0] += (P.x - c.x) + (M.x - c.x);              \
        s[1] += (P.y - c.y) + (M.y - c.y);              \
        s[2] += (P.z - c.z) + (M.z - c.z);              \
        s[3] += (P.w - c.w) + (M.w - c.w);              \
    }

template <int ND>
__global__ void __launch_bounds__(256, ND == 2 ? 4 : 3) acoustic_step_kernel(const StepArgs a) {
    pdl_launch_dependents();
    const Layout &L = a.L;
    const int tid = threadIdx.y * 32 + threadIdx.x;
    pdl_wait();
    const unsigned lin_block = blockIdx.x;
    sample_points(a, lin_block, 256, tid);
    const unsigned bx = lin_block % a.gx, byz = lin_block / a.gx;
    const unsigned by = byz % a.gy, bz = byz / a.gy;

    const int jz = (bx * 32 + threadIdx.x) * 4;
    int jx, jy;
    if (ND == 2) { jx = by * 8 + threadIdx.y; jy = 0; }
    else { jy = by * 8 + threadIdx.y; jx = bz; }
    if (jz >= L.Pz || jx >= L.Px || jy >= L.Py) return;
    const int ix = jx - L.nb, iy = jy - L.nby, iz = jz - L.nbz;
    const bool phys = a.PZ != nullptr && ix >= 0 && ix < L.nx && iy >= 0 && iy < L.ny && iz >= 0 && iz < L.nz;
    const long long po = ((long long)ix * L.ny + iy) * L.upz + iz;
    // measured (per-step fused, fraction of the HBM roofline): c4 0.708 -> 0.725 with the prefetch; c1 0.768 -> 0.666 (the 2D
    // fields live in L2 and the early plane lines compete with them), so 3D only; TTI 2D 0.575 -> 0.549: not used there either
    if (ND == 3 && phys) prefetch_planes(a.PZ + po, L.Nu, a.r);

    const long long off = L.org + jx * L.sx + jy * L.sy + jz;
    const float *uc = a.u0 + off;
    const float4 c = ld4(uc);
    const float4 zm = ld4(uc - 4), zp = ld4(uc + 4);
    const float win[12] = {zm.x, zm.y, zm.z, zm.w, c.x, c.y, c.z, c.w, zp.x, zp.y, zp.z, zp.w};
    const float cc[4] = {c.x, c.y, c.z, c.w};

    float lap[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
    for (int j = 4; j >= 1; j--) {   // small weights first
        float s[4];
#pragma unroll
        for (int q = 0; q < 4; q++) s[q] = (win[4 + q + j] - cc[q]) + (win[4 + q - j] - cc[q]);
        {
            const float4 P = ld4(uc + j * L.sx), M = ld4(uc - j * L.sx);
            ACC_AXIS(P, M)
        }
        if (ND == 3) {
            const float4 P = ld4(uc + j * L.sy), M = ld4(uc - j * L.sy);
            ACC_AXIS(P, M)
        }
        const float w = w2(j);
#pragma unroll
        for (int q = 0; q < 4; q++) lap[q] = fmaf(w, s[q], lap[q]);
    }

    const float4 k24 = ld4(a.K2 + off);
    const float k2[4] = {k24.x, k24.y, k24.z, k24.w};
    float sxy = a.dampx[jx];
    if (ND == 3) sxy += a.dampy[jy];
    const float4 dz4 = ld4(a.dampz + jz);
    const float dzv[4] = {dz4.x, dz4.y, dz4.z, dz4.w};
    const float4 du4 = ld4(a.d0 + off);
    const float du[4] = {du4.x, du4.y, du4.z, du4.w};

    float inj[4] = {0.f, 0.f, 0.f, 0.f};
    if (jx >= a.bx0 && jx <= a.bx1 && jy >= a.by0 && jy <= a.by1 && jz + 3 >= a.bz0 && jz <= a.bz1)
        inject_quad(a, (long long)jx * L.Py + jy, jz, k2, inj);

    float dn[4], un[4];
#pragma unroll
    for (int q = 0; q < 4; q++) {
        const float k1 = k1_of(sxy + dzv[q]);
        float d = fmaf(k1, du[q], k2[q] * lap[q]) + inj[q];
        float u = cc[q] + d;
        const bool in = (jz + q) < L.Pz;
        dn[q] = in ? d : 0.0f;
        un[q] = in ? u : 0.0f;
    }
    st4(a.d0 + off, make_float4(dn[0], dn[1], dn[2], dn[3]));
    const float4 unew = make_float4(un[0], un[1], un[2], un[3]);
    st4(a.n0 + off, unew);

    if (phys) probe_quad<(ND == 2 ? 1 : 2)>(a.PZ + po, L.Nu, a.Zrow, a.r, unew);
}

}  // namespace rtm

