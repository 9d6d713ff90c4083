// tti3d.cuh -- 3D pseudo-acoustic TTI time step ("TTI", L81 "generalize to 3D"; reading
// C30) with fused damping, injection, deferred sampling and probing of the single field (p + r)/2.
//
//   symmetry axis  n  = (sin th cos ph, sin th sin ph, cos th);   e1 = (cos th cos ph, cos th sin ph, -sin th),
//   e2 = (-sin ph, cos ph, 0): an orthonormal basis of the plane perpendicular to it.
//   G_v f = v . (Dx f, Dy f, Dz f), D = undivided centred order-8 first derivative; g is evaluated on P, zero outside
//   (cos = sin = 0 in the coefficient halo does that).
//   H_par  f = -G_n^T G_n f                      = Dx(nx g) + Dy(ny g) + Dz(nz g),                    g  = G_n f
//   H_perp f = -(G_e1^T G_e1 + G_e2^T G_e2) f    = Dx(e1x g1 + e2x g2) + Dy(e1y g1 + e2y g2) + Dz(e1z g1),  g1, g2 = G_e1 f, G_e2 f
//   forward (post-mix):  A = H_perp p, B = H_par r,  dp' = K1 dp + K2 (epsh A + delh B),  dr' = K1 dr + K2 (delh A + B)
//   adjoint (pre-mix):   a = epsh p + delh r, b = delh p + r,  dp' = K1 dp + K2 H_perp a,  dr' = K1 dr + K2 H_par b
//
// Three kernels per step, the six intermediate vector components in global memory (L2 keeps the 9 planes a block row
// needs):
//   tti3d_mix_kernel  (adjoint only)  a, b -> the two "new field" buffers, which are free until the step kernel writes them;
//   tti3d_grad_kernel                 (fa, fb) -> F[0..2] = (e1x g1 + e2x g2, e1y g1 + e2y g2, e1z g1),  F[3..5] = (nx, ny, nz) g;
//   tti3d_step_kernel<TM>             A = Dx F0 + Dy F1 + Dz F2, B = Dx F3 + Dy F4 + Dz F5, update, inject, sample, probe.
// Thread = one z-quad of one (jx, jy) row; block 32 x 8 (128 z points x 8 rows), grid (z blocks, y blocks, planes).
// A first, correct version: HBM-bound at ~30 array passes per step; not yet tiled in shared memory.
#pragma once
#include "common.cuh"

namespace rtm {

// undivided centred order-8 first derivatives of the quad at p: along an axis with stride s (x, y) ...
__device__ __forceinline__ void d1_strided(const float *__restrict__ p, long long s, float out[4]) {
    out[0] = out[1] = out[2] = out[3] = 0.f;
#pragma unroll
    for (int j = 4; j >= 1; j--) {   // small weights first
        const float w = w1(j);
        const float4 P = ld4(p + j * s), M = ld4(p - j * s);
        out[0] = fmaf(w, P.x - M.x, out[0]); out[1] = fmaf(w, P.y - M.y, out[1]);
        out[2] = fmaf(w, P.z - M.z, out[2]); out[3] = fmaf(w, P.w - M.w, out[3]);
    }
}
// ... and along z (contiguous): a window of 12 floats around the quad
__device__ __forceinline__ void d1_z(const float *__restrict__ p, float out[4]) {
    const float4 m = ld4(p - 4), c = ld4(p), q = ld4(p + 4);
    const float w[12] = {m.x, m.y, m.z, m.w, c.x, c.y, c.z, c.w, q.x, q.y, q.z, q.w};
#pragma unroll
    for (int e = 0; e < 4; e++) {
        float acc = 0.f;
#pragma unroll
        for (int j = 4; j >= 1; j--) acc = fmaf(w1(j), w[4 + e + j] - w[4 + e - j], acc);
        out[e] = acc;
    }
}

// thread -> (jx, jy, jz); false if the quad lies outside the (internal) padded grid
__device__ __forceinline__ bool tti3d_quad(const StepArgs &a, unsigned lin_block, int &jx, int &jy, int &jz) {
    const unsigned bx = lin_block % a.gx, byz = lin_block / a.gx;
    jz = (bx * 32 + threadIdx.x) * 4;
    jy = (byz % a.gy) * 8 + threadIdx.y;
    jx = byz / a.gy;
    return jz < a.L.Pz && jy < a.L.Py && jx < a.L.Px;
}

// adjoint pre-mix (O6): a = epsh p + delh r, b = delh p + r on P -> n0, n1 (halo untouched: it stays zero)
__global__ void __launch_bounds__(256) tti3d_mix_kernel(const StepArgs a) {
    pdl_launch_dependents();
    pdl_wait();
    int jx, jy, jz;
    if (!tti3d_quad(a, blockIdx.x, jx, jy, jz)) return;
    const long long o = a.L.org + jx * a.L.sx + jy * a.L.sy + jz;
    const float4 p = ld4(a.u0 + o), r = ld4(a.u1 + o), e = ld4(a.epsh + o), d = ld4(a.delh + o);
    float4 ma, mb;
    ma.x = fmaf(e.x, p.x, d.x * r.x); mb.x = fmaf(d.x, p.x, r.x);
    ma.y = fmaf(e.y, p.y, d.y * r.y); mb.y = fmaf(d.y, p.y, r.y);
    ma.z = fmaf(e.z, p.z, d.z * r.z); mb.z = fmaf(d.z, p.z, r.z);
    ma.w = fmaf(e.w, p.w, d.w * r.w); mb.w = fmaf(d.w, p.w, r.w);
    st4(a.n0 + o, ma);     // epsh = delh = 0 outside P (coefficient halo and the ragged lanes of the last quad): zeros stay zeros
    st4(a.n1 + o, mb);
}

// rotated gradients times the direction vectors: F[0..2] feed H_perp, F[3..5] feed H_par
__global__ void __launch_bounds__(256) tti3d_grad_kernel(const StepArgs a) {
    pdl_launch_dependents();
    pdl_wait();
    int jx, jy, jz;
    if (!tti3d_quad(a, blockIdx.x, jx, jy, jz)) return;
    const Layout &L = a.L;
    const long long o = L.org + jx * L.sx + jy * L.sy + jz;
    const float *fa = (a.adjoint ? a.n0 : a.u0) + o, *fb = (a.adjoint ? a.n1 : a.u1) + o;
    float ax[4], ay[4], az[4], bx[4], by[4], bz[4];
    d1_strided(fa, L.sx, ax); d1_strided(fa, L.sy, ay); d1_z(fa, az);
    d1_strided(fb, L.sx, bx); d1_strided(fb, L.sy, by); d1_z(fb, bz);
    const float4 ct4 = ld4(a.cs + o), st4_ = ld4(a.sn + o), cp4 = ld4(a.cp + o), sp4 = ld4(a.sp + o);
    const float ct[4] = {ct4.x, ct4.y, ct4.z, ct4.w}, st[4] = {st4_.x, st4_.y, st4_.z, st4_.w};
    const float cp[4] = {cp4.x, cp4.y, cp4.z, cp4.w}, sp[4] = {sp4.x, sp4.y, sp4.z, sp4.w};
    float F[6][4];
#pragma unroll
    for (int e = 0; e < 4; e++) {
        const float nx = st[e] * cp[e], ny = st[e] * sp[e], nz = ct[e];
        const float e1x = ct[e] * cp[e], e1y = ct[e] * sp[e], e1z = -st[e], e2x = -sp[e], e2y = cp[e];
        const float g1 = fmaf(e1z, az[e], fmaf(e1y, ay[e], e1x * ax[e]));
        const float g2 = fmaf(e2y, ay[e], e2x * ax[e]);
        const float gn = fmaf(nz, bz[e], fmaf(ny, by[e], nx * bx[e]));
        F[0][e] = fmaf(e2x, g2, e1x * g1);
        F[1][e] = fmaf(e2y, g2, e1y * g1);
        F[2][e] = e1z * g1;
        F[3][e] = nx * gn;
        F[4][e] = ny * gn;
        F[5][e] = nz * gn;
    }
#pragma unroll
    for (int k = 0; k < 6; k++) st4(a.F[k] + o, make_float4(F[k][0], F[k][1], F[k][2], F[k][3]));
}

template <int TM, bool TWO = false>
__global__ void __launch_bounds__(256, 2) tti3d_step_kernel(const StepArgs a) {
    pdl_launch_dependents();
    pdl_wait();
    const Layout &L = a.L;
    const int tid = threadIdx.y * 32 + threadIdx.x;
    sample_points(a, blockIdx.x, 256, tid);
    int jx, jy, jz;
    if (!tti3d_quad(a, blockIdx.x, jx, jy, jz)) return;
    const long long off = L.org + jx * L.sx + jy * L.sy + jz;
    float A[4], B[4];
    {
        float dx[4], dy[4], dz[4];
        d1_strided(a.F[0] + off, L.sx, dx); d1_strided(a.F[1] + off, L.sy, dy); d1_z(a.F[2] + off, dz);
#pragma unroll
        for (int q = 0; q < 4; q++) A[q] = (dx[q] + dy[q]) + dz[q];
        d1_strided(a.F[3] + off, L.sx, dx); d1_strided(a.F[4] + off, L.sy, dy); d1_z(a.F[5] + off, dz);
#pragma unroll
        for (int q = 0; q < 4; q++) B[q] = (dx[q] + dy[q]) + dz[q];
    }
    const float4 p4 = ld4(a.u0 + off), r4 = ld4(a.u1 + off), dp4 = ld4(a.d0 + off), dr4 = ld4(a.d1 + off), k24 = ld4(a.K2 + off);
    const float pc[4] = {p4.x, p4.y, p4.z, p4.w}, rc[4] = {r4.x, r4.y, r4.z, r4.w};
    const float dp[4] = {dp4.x, dp4.y, dp4.z, dp4.w}, dr[4] = {dr4.x, dr4.y, dr4.z, dr4.w};
    const float k2[4] = {k24.x, k24.y, k24.z, k24.w};
    float eh[4] = {1.f, 1.f, 1.f, 1.f}, dh[4] = {0.f, 0.f, 0.f, 0.f};
    if (!a.adjoint) {
        const float4 e4 = ld4(a.epsh + off), d4 = ld4(a.delh + off);
        eh[0] = e4.x; eh[1] = e4.y; eh[2] = e4.z; eh[3] = e4.w;
        dh[0] = d4.x; dh[1] = d4.y; dh[2] = d4.z; dh[3] = d4.w;
    }
    const float sxy = a.dampx[jx] + a.dampy[jy];
    const float4 dz4 = ld4(a.dampz + jz);
    const float dzv[4] = {dz4.x, dz4.y, dz4.z, dz4.w};

    float inj[4] = {0.f, 0.f, 0.f, 0.f};
    if (jx >= a.bx0 && jx <= a.bx1 && jy >= a.by0 && jy <= a.by1 && jz + 3 >= a.bz0 && jz <= a.bz1)
        inject_quad(a, (long long)jx * L.Py + jy, jz, k2, inj);

    float pn[4], rn[4], dpn[4], drn[4], pr[4];
#pragma unroll
    for (int q = 0; q < 4; q++) {
        const float k1 = k1_of(sxy + dzv[q]);
        const float ra = a.adjoint ? A[q] : fmaf(eh[q], A[q], dh[q] * B[q]);
        const float rb = a.adjoint ? B[q] : fmaf(dh[q], A[q], B[q]);
        const float d0 = fmaf(k1, dp[q], k2[q] * ra) + inj[q];
        const float d1 = fmaf(k1, dr[q], k2[q] * rb) + inj[q];
        const bool in = (jz + q) < L.Pz;
        dpn[q] = in ? d0 : 0.f;
        drn[q] = in ? d1 : 0.f;
        pn[q] = in ? pc[q] + d0 : 0.f;
        rn[q] = in ? rc[q] + d1 : 0.f;
        pr[q] = 0.5f * (pn[q] + rn[q]);
    }
    st4(a.d0 + off, make_float4(dpn[0], dpn[1], dpn[2], dpn[3]));
    st4(a.d1 + off, make_float4(drn[0], drn[1], drn[2], drn[3]));
    st4(a.n0 + off, make_float4(pn[0], pn[1], pn[2], pn[3]));
    st4(a.n1 + off, make_float4(rn[0], rn[1], rn[2], rn[3]));

    const int ix = jx - L.nb, iy = jy - L.nby, iz = jz - L.nbz;
    if (ix >= 0 && ix < L.nx && iy >= 0 && iy < L.ny && iz >= 0 && iz < L.nz) {
        const long long o = ((long long)ix * L.ny + iy) * L.upz + iz;
        if (!TWO) {
            const float4 v = make_float4(pr[0], pr[1], pr[2], pr[3]);
            if (TM > 0) { if (a.hist != nullptr) stcs4(a.hist + o, v); }
            else if (a.PZ != nullptr) probe_quad<2>(a.PZ + o, L.Nu, a.Zrow, a.r, v);
        } else {
            // p and r probed apart (readings C29 + C30), laid out as in tti.cuh: plane (or history half-slot) 2k = p, 2k + 1 = r
            const float4 wp = make_float4(pn[0], pn[1], pn[2], pn[3]), wr = make_float4(rn[0], rn[1], rn[2], rn[3]);
            if (TM > 0) {
                if (a.hist != nullptr) { stcs4(a.hist + o, wp); stcs4(a.hist + L.Nu + o, wr); }
            } else if (a.PZ != nullptr) {
                for (int f = 0; f < 2; f++) probe_quad<2>(a.PZ + (long long)f * L.Nu + o, 2 * L.Nu, a.Zrow, a.r, f ? wr : wp);
            }
        }
    }
}

}  // namespace rtm
