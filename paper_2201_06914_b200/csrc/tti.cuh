// tti.cuh -- 2D pseudo-acoustic TTI time step (a2) with fused damping, injection, deferred sampling
// and probe accumulation of the single field (p + r)/2 (reading C10).
//
//   forward (post-mix, O5):  A = H_perp p, B = H_par r,
//        dp_new = K1 dp + K2 (epsh A + delh B),  dr_new = K1 dr + K2 (delh A + B)
//   adjoint (pre-mix, O6):   a = epsh p + delh r, b = delh p + r, A = H_perp a, B = H_par b,
//        dp_new = K1 dp + K2 A,                  dr_new = K1 dr + K2 B
//   H_perp f = Dx(cos g) - Dz(sin g), g = cos Dx f - sin Dz f ;  H_par f = Dx(sin g) + Dz(cos g),
//   g = sin Dx f + cos Dz f ; D = undivided centred order-8 first derivative; g is zero outside P
//   (cos = sin = 0 in the coefficient halo does that).
//
// Two-stage tile kernel: stage 1 loads the (mixed) fields with a halo of 8 into shared memory,
// stage 2 forms the four products cos g_perp, sin g_perp, sin g_par, cos g_par on the tile + halo 4,
// stage 3 differentiates them.  Tile = 16 (x) x 64 (z), 256 threads, one z-quad per thread.
#pragma once
#include "common.cuh"

namespace rtm {

constexpr int TTI_TZ = 64;
constexpr int TTI_FZ = TTI_TZ + 16;   // field tile (halo 8)
constexpr int TTI_GZ = TTI_TZ + 8;    // product tile (halo 4)
// Rows per tile: 16 (256 threads) or 32 (512 threads).  The halo recompute falls from 2.5 x / 1.69 x of the tile in stages
// 1 / 2 to 1.875 x / 1.41 x with 32 rows, at the same 32 warps per SM (2 blocks of 512 threads and 77 KB instead of 4
// blocks of 256 threads and 48 KB); the per-step fused variant (80 registers for the probe pipeline) keeps 16 rows.
__host__ __device__ constexpr int tti_smem(int tx) { return (2 * (tx + 16) * TTI_FZ + 4 * (tx + 8) * TTI_GZ) * 4; }

template <int TM, bool TWO = false, int TTI_TX = 16>
__global__ void __launch_bounds__(16 * TTI_TX, TM == 0 ? 3 : (TTI_TX == 16 ? 4 : 2)) tti_step_kernel(const StepArgs a) {
    constexpr int TTI_FX = TTI_TX + 16, TTI_GX = TTI_TX + 8, NT = 16 * TTI_TX;
    extern __shared__ __align__(16) float smem[];
    float *sA = smem;                          // [FX][FZ]
    float *sB = sA + TTI_FX * TTI_FZ;
    float *P1 = sB + TTI_FX * TTI_FZ;          // cos g_perp  [GX][GZ]
    float *P2 = P1 + TTI_GX * TTI_GZ;          // sin g_perp
    float *P3 = P2 + TTI_GX * TTI_GZ;          // sin g_par
    float *P4 = P3 + TTI_GX * TTI_GZ;          // cos g_par

    const Layout &L = a.L;
    const int tid = threadIdx.y * 16 + threadIdx.x;
    if (TM == 0) pdl_launch_dependents();
    if (TM > 0 && blockIdx.x < (unsigned)a.fl_blocks) {
        pdl_launch_dependents();
        flush_role<(TM > 0 ? TM : 1)>(a, smem, tid, NT, blockIdx.x);
        return;
    }
    pdl_wait();
    if (TM > 0) pdl_launch_dependents();   // only now: lets the next step's flush role run without a wait (see flush_role)
    const unsigned lin_block = blockIdx.x - (TM > 0 ? a.fl_blocks : 0);
    sample_points(a, lin_block, NT, tid);

    const int z0 = (lin_block % a.gx) * TTI_TZ, x0 = (lin_block / a.gx) * TTI_TX;

    // ---- stage 1: (mixed) fields, halo 8 ----
    // All loads of a thread's N1 quads are issued before the first one is used: the stage is a single round trip to
    // L2 / DRAM per block instead of one per loop iteration (the fields do not all stay in L2 beside the probe stream).
    constexpr int N1 = (TTI_FX * (TTI_FZ / 4) + NT - 1) / NT;
    {
        float4 va[N1], vb[N1], ve[N1], vd[N1];
        int so[N1];
#pragma unroll
        for (int k = 0; k < N1; k++) {
            const int i = tid + k * NT;
            const int lx = i / (TTI_FZ / 4), lq = i % (TTI_FZ / 4);
            const int jx = x0 - 8 + lx, jz = z0 - 8 + lq * 4;
            so[k] = i < TTI_FX * (TTI_FZ / 4) ? lx * TTI_FZ + lq * 4 : -1;
            va[k] = make_float4(0.f, 0.f, 0.f, 0.f); vb[k] = va[k]; ve[k] = va[k]; vd[k] = va[k];
            if (so[k] >= 0 && jx < L.Px + 8 && jz + 3 < L.pz - 8) {
                const long long o = L.org + jx * L.sx + jz;
                va[k] = ld4(a.u0 + o);
                vb[k] = ld4(a.u1 + o);
                if (a.adjoint) { ve[k] = ld4(a.epsh + o); vd[k] = ld4(a.delh + o); }
            }
        }
#pragma unroll
        for (int k = 0; k < N1; k++) {
            if (so[k] < 0) continue;
            float4 xa = va[k], xb = vb[k];
            if (a.adjoint) {
                const float4 e = ve[k], d = vd[k];
                float4 ma, mb;
                ma.x = fmaf(e.x, xa.x, d.x * xb.x); mb.x = fmaf(d.x, xa.x, xb.x);
                ma.y = fmaf(e.y, xa.y, d.y * xb.y); mb.y = fmaf(d.y, xa.y, xb.y);
                ma.z = fmaf(e.z, xa.z, d.z * xb.z); mb.z = fmaf(d.z, xa.z, xb.z);
                ma.w = fmaf(e.w, xa.w, d.w * xb.w); mb.w = fmaf(d.w, xa.w, xb.w);
                xa = ma; xb = mb;
            }
            st4(sA + so[k], xa);
            st4(sB + so[k], xb);
        }
    }
    // cos / sin of this thread's stage-2 quads: requested before the barrier, so that their latency overlaps with it
    constexpr int N2 = (TTI_GX * (TTI_GZ / 4) + NT - 1) / NT;
    float4 csv[N2], snv[N2];
#pragma unroll
    for (int k = 0; k < N2; k++) {
        const int i = tid + k * NT;
        const int lx = i / (TTI_GZ / 4), lq = i - lx * (TTI_GZ / 4);
        const int jx = x0 - 4 + lx, jz = z0 - 4 + lq * 4;
        csv[k] = make_float4(0.f, 0.f, 0.f, 0.f); snv[k] = csv[k];
        if (i < TTI_GX * (TTI_GZ / 4) && jx < L.Px + 8 && jz + 3 < L.pz - 8) {
            const long long o = L.org + jx * L.sx + jz;
            csv[k] = ld4(a.cs + o);
            snv[k] = ld4(a.sn + o);
        }
    }
    __syncthreads();

    // ---- stage 2: rotated gradients times cos / sin, halo 4; one z-quad per thread and round ----
    // centred first derivative of a quad: x from the 8 neighbour rows (LDS.128 each), z from the 12-float window
#pragma unroll
    for (int k = 0; k < N2; k++) {
        const int i = tid + k * NT;
        if (i >= TTI_GX * (TTI_GZ / 4)) break;
        const int lx = i / (TTI_GZ / 4), lq = i - lx * (TTI_GZ / 4);
        const float4 cs4 = csv[k], sn4 = snv[k];
        const float *fa = sA + (lx + 4) * TTI_FZ + (lq * 4 + 4);
        const float *fb = sB + (lx + 4) * TTI_FZ + (lq * 4 + 4);
        float ax[4] = {0.f, 0.f, 0.f, 0.f}, bx[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int j = 4; j >= 1; j--) {
            const float w = w1(j);
            const float4 pa = ld4(fa + j * TTI_FZ), ma = ld4(fa - j * TTI_FZ);
            const float4 pb = ld4(fb + j * TTI_FZ), mb = ld4(fb - j * TTI_FZ);
            ax[0] = fmaf(w, pa.x - ma.x, ax[0]); ax[1] = fmaf(w, pa.y - ma.y, ax[1]);
            ax[2] = fmaf(w, pa.z - ma.z, ax[2]); ax[3] = fmaf(w, pa.w - ma.w, ax[3]);
            bx[0] = fmaf(w, pb.x - mb.x, bx[0]); bx[1] = fmaf(w, pb.y - mb.y, bx[1]);
            bx[2] = fmaf(w, pb.z - mb.z, bx[2]); bx[3] = fmaf(w, pb.w - mb.w, bx[3]);
        }
        const float4 am = ld4(fa - 4), ac = ld4(fa), ap = ld4(fa + 4);
        const float4 bm = ld4(fb - 4), bc = ld4(fb), bp = ld4(fb + 4);
        const float wa[12] = {am.x, am.y, am.z, am.w, ac.x, ac.y, ac.z, ac.w, ap.x, ap.y, ap.z, ap.w};
        const float wb[12] = {bm.x, bm.y, bm.z, bm.w, bc.x, bc.y, bc.z, bc.w, bp.x, bp.y, bp.z, bp.w};
        const float cs[4] = {cs4.x, cs4.y, cs4.z, cs4.w}, sn[4] = {sn4.x, sn4.y, sn4.z, sn4.w};
        float o1[4], o2[4], o3[4], o4[4];
#pragma unroll
        for (int e = 0; e < 4; e++) {
            float az = 0.f, bz = 0.f;
#pragma unroll
            for (int j = 4; j >= 1; j--) {
                const float w = w1(j);
                az = fmaf(w, wa[4 + e + j] - wa[4 + e - j], az);
                bz = fmaf(w, wb[4 + e + j] - wb[4 + e - j], bz);
            }
            const float gp = cs[e] * ax[e] - sn[e] * az;   // g_perp
            const float gl = sn[e] * bx[e] + cs[e] * bz;   // g_par
            o1[e] = cs[e] * gp;
            o2[e] = sn[e] * gp;
            o3[e] = sn[e] * gl;
            o4[e] = cs[e] * gl;
        }
        const int g = lx * TTI_GZ + lq * 4;
        st4(P1 + g, make_float4(o1[0], o1[1], o1[2], o1[3]));
        st4(P2 + g, make_float4(o2[0], o2[1], o2[2], o2[3]));
        st4(P3 + g, make_float4(o3[0], o3[1], o3[2], o3[3]));
        st4(P4 + g, make_float4(o4[0], o4[1], o4[2], o4[3]));
    }
    // stage-3 operands are requested BEFORE the barrier, so that their L2 latency overlaps with the barrier wait
    // and the shared-memory arithmetic of stage 3 instead of sitting in front of the update
    const int lx = threadIdx.y, lz = threadIdx.x * 4;
    const int jx = x0 + lx, jz = z0 + lz;
    const bool act3 = jx < L.Px && jz < L.Pz;
    const long long off = L.org + jx * L.sx + jz;
    float4 p4 = make_float4(0.f, 0.f, 0.f, 0.f), r4 = p4, dp4 = p4, dr4 = p4, k24 = p4, e4 = p4, d4 = p4;
    if (act3) {
        p4 = ld4(a.u0 + off); r4 = ld4(a.u1 + off);
        dp4 = ld4(a.d0 + off); dr4 = ld4(a.d1 + off);
        k24 = ld4(a.K2 + off);
        if (!a.adjoint) { e4 = ld4(a.epsh + off); d4 = ld4(a.delh + off); }
    }
    __syncthreads();

    // ---- stage 3: second derivative pass, update, inject, probe ----
    if (!act3) return;

    float A[4], B[4];
    {
        const int g = (lx + 4) * TTI_GZ + (lz + 4);
        float dx1[4] = {0.f, 0.f, 0.f, 0.f}, dx3[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int j = 4; j >= 1; j--) {
            const float w = w1(j);
            const float4 p1 = ld4(P1 + g + j * TTI_GZ), m1 = ld4(P1 + g - j * TTI_GZ);
            const float4 p3 = ld4(P3 + g + j * TTI_GZ), m3 = ld4(P3 + g - j * TTI_GZ);
            dx1[0] = fmaf(w, p1.x - m1.x, dx1[0]); dx1[1] = fmaf(w, p1.y - m1.y, dx1[1]);
            dx1[2] = fmaf(w, p1.z - m1.z, dx1[2]); dx1[3] = fmaf(w, p1.w - m1.w, dx1[3]);
            dx3[0] = fmaf(w, p3.x - m3.x, dx3[0]); dx3[1] = fmaf(w, p3.y - m3.y, dx3[1]);
            dx3[2] = fmaf(w, p3.z - m3.z, dx3[2]); dx3[3] = fmaf(w, p3.w - m3.w, dx3[3]);
        }
        const float4 m2 = ld4(P2 + g - 4), c2 = ld4(P2 + g), p2 = ld4(P2 + g + 4);
        const float4 m4 = ld4(P4 + g - 4), c4 = ld4(P4 + g), p4q = ld4(P4 + g + 4);
        const float w2a[12] = {m2.x, m2.y, m2.z, m2.w, c2.x, c2.y, c2.z, c2.w, p2.x, p2.y, p2.z, p2.w};
        const float w4a[12] = {m4.x, m4.y, m4.z, m4.w, c4.x, c4.y, c4.z, c4.w, p4q.x, p4q.y, p4q.z, p4q.w};
#pragma unroll
        for (int q = 0; q < 4; q++) {
            float dz2 = 0.f, dz4 = 0.f;
#pragma unroll
            for (int j = 4; j >= 1; j--) {
                const float w = w1(j);
                dz2 = fmaf(w, w2a[4 + q + j] - w2a[4 + q - j], dz2);
                dz4 = fmaf(w, w4a[4 + q + j] - w4a[4 + q - j], dz4);
            }
            A[q] = dx1[q] - dz2;
            B[q] = dx3[q] + dz4;
        }
    }

    const float pc[4] = {p4.x, p4.y, p4.z, p4.w}, rc[4] = {r4.x, r4.y, r4.z, r4.w};
    const float dp[4] = {dp4.x, dp4.y, dp4.z, dp4.w}, dr[4] = {dr4.x, dr4.y, dr4.z, dr4.w};
    const float k2[4] = {k24.x, k24.y, k24.z, k24.w};
    float eh[4] = {1.f, 1.f, 1.f, 1.f}, dh[4] = {0.f, 0.f, 0.f, 0.f};
    if (!a.adjoint) {
        eh[0] = e4.x; eh[1] = e4.y; eh[2] = e4.z; eh[3] = e4.w;
        dh[0] = d4.x; dh[1] = d4.y; dh[2] = d4.z; dh[3] = d4.w;
    }
    const float sx = a.dampx[jx];
    const float4 dz4 = ld4(a.dampz + jz);
    const float dzv[4] = {dz4.x, dz4.y, dz4.z, dz4.w};

    float inj[4] = {0.f, 0.f, 0.f, 0.f};
    if (jx >= a.bx0 && jx <= a.bx1 && jz + 3 >= a.bz0 && jz <= a.bz1) inject_quad(a, jx, jz, k2, inj);

    float pn[4], rn[4], dpn[4], drn[4], pr[4];
#pragma unroll
    for (int q = 0; q < 4; q++) {
        const float k1 = k1_of(sx + dzv[q]);
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

    if (TM > 0 ? (a.hist != nullptr) : (a.PZ != nullptr)) {
        const int ix = jx - L.nb, iz = jz - L.nbz;
        if (ix >= 0 && ix < L.nx && iz >= 0 && iz < L.nz) {
            const long long o = (long long)ix * L.upz + iz;
            const float4 v = make_float4(pr[0], pr[1], pr[2], pr[3]);
            if (!TWO) {
                if (TM > 0) stcs4(a.hist + o, v);
                else probe_quad<2>(a.PZ + o, L.Nu, a.Zrow, a.r, v);
            } else {
                // four compressed arrays for the TTI gradient (PAPER.md:L39-45 on the (p, r) system of L77; reading
                // C29): p and r probed apart with the same row of Z; plane (or history half-slot) 2k = p, 2k + 1 = r
                const float4 wp = make_float4(pn[0], pn[1], pn[2], pn[3]), wr = make_float4(rn[0], rn[1], rn[2], rn[3]);
                if (TM > 0) {
                    stcs4(a.hist + o, wp);
                    stcs4(a.hist + L.Nu + o, wr);
                } else {
                    for (int f = 0; f < 2; f++)
                        probe_quad<2>(a.PZ + (long long)f * L.Nu + o, 2 * L.Nu, a.Zrow, a.r, f ? wr : wp);
                }
            }
        }
    }
}

}  // namespace rtm
