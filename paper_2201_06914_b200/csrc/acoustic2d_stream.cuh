// acoustic2d_stream.cuh -- 2D isotropic acoustic time step (a1) for time-blocked probing, register-blocked
// streaming along the slow axis (x).  Fused: damping, source injection (a3), deferred receiver sampling
// (a4), history store for the probe (a5) and, in the leading blocks of the launch, the flush role that
// applies T rows of Z to the previous time block's history.
//
// Thread = one z-quad column segment of RX consecutive rows.  The 9 x-neighbour quads live in a register
// queue that slides one row per iteration (1 new LDG.128 of u per row instead of 8); the two z-halo
// quads of the centre row come from L1.  Software-pipelined by hand: the five LDG.128 of row rr+1 are
// issued before the ~170 flops of row rr, so one L2 latency is exposed per thread instead of RX.
//
// Everything that does not depend on the previous step is done BEFORE griddepcontrol.wait, i.e. while
// the previous step's grid is still draining (programmatic dependent launch): the injection amounts of
// this thread's rows (row-CSR lookup -> shared memory), the sampling tables, the Z rows of the flush role.
//
// K1 = (1-s)/(1+s), s = sx + sz: interior rows/quads take K1 = 1 exactly; layer points with one active
// axis read the per-axis table k1x / k1z (computed once on the device with the same IEEE division);
// only the corners of the layer divide.
#pragma once
#include "common.cuh"

namespace rtm {

// 4 blocks of 128 threads per SM = 128 registers: without the bound the compiler takes 136 - 142 and the launch loses a
// quarter of its resident blocks (measured: 12.2 us per step instead of 10.1 at c1).
template <int TM, int RX>
__global__ void __launch_bounds__(128, 4) acoustic2d_stream_kernel(const __grid_constant__ StepArgs a) {
    extern __shared__ __align__(16) float dyn_smem[];
    const Layout &L = a.L;
    const int tid = threadIdx.x;
    if (blockIdx.x < (unsigned)a.fl_blocks) {
        pdl_launch_dependents();
        // up to 16 history values as float4 per thread; 32 as float2 (register budget), two groups in flight
        if constexpr (TM <= 16) flush_role4<TM>(a, dyn_smem, tid, 128, blockIdx.x);
        else flush_role<TM, 2>(a, dyn_smem, tid, 128, blockIdx.x);
        return;
    }
    const unsigned lin_block = blockIdx.x - a.fl_blocks;
    DBG_STAMP(a, 0);   // timing experiments (dbg & 16): block start / before the wait / after it / end
    // flattened task index: (row chunk, z-quad) pairs are dealt to consecutive threads, so no lane idles
    // on a ragged Pz; a.gx = number of z-quads per row
    const unsigned task = lin_block * 128u + tid;
    const unsigned chunk = task / a.gx;
    const int jz = (int)(task - chunk * a.gx) * 4;
    const int x0 = (int)chunk * RX;
    const bool active = x0 < L.Px;

    // ---- prologue on static data (before the grid dependency is resolved) ----------------------
    // (i) deferred sampling tables of this thread's receiver
    const bool do_smp = a.smp_out != nullptr && task < (unsigned)a.nsmp;
    int sidx[4];
    float swt[4];
    if (do_smp) {
        const int4 i4 = *reinterpret_cast<const int4 *>(a.smp_idx + 4 * (size_t)task);
        const float4 w4 = ld4(a.smp_w + 4 * (size_t)task);
        sidx[0] = i4.x; sidx[1] = i4.y; sidx[2] = i4.z; sidx[3] = i4.w;
        swt[0] = w4.x; swt[1] = w4.y; swt[2] = w4.z; swt[3] = w4.w;
    }
    // (ii) injection amounts v = scale * w * val of this thread's RX quads -> smem [RX][128]; bit rr of
    // imask = row rr has something to add
    float4 *injs = reinterpret_cast<float4 *>(dyn_smem);
    unsigned imask = 0;
    if (active && jz + 3 >= a.bz0 && jz <= a.bz1 && x0 <= a.bx1 && x0 + RX - 1 >= a.bx0) {
        int rs[RX + 1];
#pragma unroll
        for (int i = 0; i <= RX; i++) rs[i] = a.row_start[min(x0 + i, L.Px)];
        int4 e0[RX];
#pragma unroll
        for (int rr = 0; rr < RX; rr++)
            if (rs[rr + 1] > rs[rr]) e0[rr] = *reinterpret_cast<const int4 *>(a.ent + rs[rr]);
        float v0[RX];
#pragma unroll
        for (int rr = 0; rr < RX; rr++)
            if (rs[rr + 1] > rs[rr]) v0[rr] = a.inj_val[e0[rr].y];
#pragma unroll
        for (int rr = 0; rr < RX; rr++) {
            if (rs[rr + 1] <= rs[rr]) continue;
            float acc[4] = {0.f, 0.f, 0.f, 0.f};
            bool any = false;
            {
                const int dz = e0[rr].x - jz;
                const float v = a.inj_scale * __int_as_float(e0[rr].z) * v0[rr];
                if (dz >= 0 && dz < 4) {
                    any = true;
#pragma unroll
                    for (int q = 0; q < 4; q++)
                        if (q == dz) acc[q] += v;
                }
            }
            for (int e = rs[rr] + 1; e < rs[rr + 1]; e++) {   // further entries of the row (off-grid points)
                const InjEntry en = a.ent[e];
                const int dz = en.jz - jz;
                if (dz >= 0 && dz < 4) {
                    const float v = a.inj_scale * en.w * a.inj_val[en.id];
                    any = true;
#pragma unroll
                    for (int q = 0; q < 4; q++)
                        if (q == dz) acc[q] += v;
                }
            }
            if (any) {
                injs[rr * 128 + tid] = make_float4(acc[0], acc[1], acc[2], acc[3]);
                imask |= 1u << rr;
            }
        }
    }
    // (iii) per-thread z tables
    float dzv[4] = {0.f, 0.f, 0.f, 0.f}, k1z[4] = {1.f, 1.f, 1.f, 1.f};
    if (active) {
        const float4 d4 = ld4(a.dampz + jz), k4 = ld4(a.k1z + jz);
        dzv[0] = d4.x; dzv[1] = d4.y; dzv[2] = d4.z; dzv[3] = d4.w;
        k1z[0] = k4.x; k1z[1] = k4.y; k1z[2] = k4.z; k1z[3] = k4.w;
    }
    const bool zdamp = (dzv[0] != 0.f) | (dzv[1] != 0.f) | (dzv[2] != 0.f) | (dzv[3] != 0.f);

    DBG_STAMP(a, 1);
    pdl_wait();   // from here on the previous step's fields are complete and visible
    DBG_STAMP(a, 2);
    // Dependents are released only now: a block of step n+1 can therefore only start once step n-1 is complete,
    // which is what lets the flush role of step n+1 skip its own wait (see flush_role4) and overlap with step n.
    pdl_launch_dependents();

    const float *__restrict__ u0 = a.u0;
    const float *__restrict__ K2 = a.K2;
    float *__restrict__ n0 = a.n0;
    float *d0 = a.d0;

    if (do_smp) {   // a4, deferred by one launch: d[j] = scale * sum_c w_c u[corner]
        float acc = 0.0f;
#pragma unroll
        for (int c = 0; c < 4; c++)
            if (swt[c] != 0.0f) acc = fmaf(swt[c], u0[sidx[c]], acc);
        a.smp_out[task] = a.smp_scale * acc;
    }
    if (active && !DBG_SKIP_STENCIL(a)) {
    const int sx = (int)L.sx;
    const int base = (int)L.org + jz;            // fsize < 2^31 (checked at create)
    const bool full = jz + 3 < L.Pz;
    const int iz = jz - L.nbz;
    const bool zphys = iz >= 0 && iz < L.nz && a.hist != nullptr;

    float4 q[8 + RX];
#pragma unroll
    for (int i = 0; i < 8; i++) q[i] = ld4(u0 + base + (x0 - 4 + i) * sx);

    // operands of the row in flight (prefetched one row ahead)
    float4 qn, zm, zp, k24, du4;
    float sxd, k1x;
    {
        const int off = base + x0 * sx;
        qn = ld4(u0 + off + 4 * sx);
        zm = ld4(u0 + off - 4);
        zp = ld4(u0 + off + 4);
        k24 = ld4(K2 + off);
        du4 = ld4(d0 + off);
        sxd = a.dampx[x0];
        k1x = a.k1x[x0];
    }

#pragma unroll
    for (int rr = 0; rr < RX; rr++) {
        const int jx = x0 + rr;
        const bool valid = jx < L.Px;
        const int off = base + jx * sx;
        q[8 + rr] = qn;
        const float4 c = q[4 + rr];
        const float win[12] = {zm.x, zm.y, zm.z, zm.w, c.x, c.y, c.z, c.w, zp.x, zp.y, zp.z, zp.w};
        const float k2[4] = {k24.x, k24.y, k24.z, k24.w};
        const float du[4] = {du4.x, du4.y, du4.z, du4.w};
        const float sxc = sxd, k1xc = k1x;
        if (rr + 1 < RX && jx + 1 < L.Px) {   // prefetch row rr+1 before the arithmetic of row rr
            const int offn = off + sx;
            qn = ld4(u0 + offn + 4 * sx);
            zm = ld4(u0 + offn - 4);
            zp = ld4(u0 + offn + 4);
            k24 = ld4(K2 + offn);
            du4 = ld4(d0 + offn);
            sxd = a.dampx[jx + 1];
            k1x = a.k1x[jx + 1];
        }
        if (!valid) continue;
        const float cc[4] = {c.x, c.y, c.z, c.w};
        // Laplacian in the difference form, two z points per instruction (FADD2 / FFMA2); the same operations in the
        // same order per point as the scalar kernels: s = (z part + x part), lap = fma(w, s, lap), small weights first
        const f32x2 clo = pk(c.x, c.y), chi = pk(c.z, c.w);
        f32x2 llo = pk(0.f, 0.f), lhi = llo;
#pragma unroll
        for (int j = 4; j >= 1; j--) {
            const float4 P = q[4 + rr + j], M = q[4 + rr - j];
            const f32x2 xlo = dd2(pk(P.x, P.y), pk(M.x, M.y), clo), xhi = dd2(pk(P.z, P.w), pk(M.z, M.w), chi);
            f32x2 zlo, zhi;
            if (j % 2 == 0) {   // shifted z windows are register-pair aligned for even shifts only
                zlo = dd2(pk(win[4 + j], win[5 + j]), pk(win[4 - j], win[5 - j]), clo);
                zhi = dd2(pk(win[6 + j], win[7 + j]), pk(win[6 - j], win[7 - j]), chi);
            } else {
                float zs[4];
#pragma unroll
                for (int e = 0; e < 4; e++) zs[e] = (win[4 + e + j] - cc[e]) + (win[4 + e - j] - cc[e]);
                zlo = pk(zs[0], zs[1]);
                zhi = pk(zs[2], zs[3]);
            }
            const float w = w2(j);
            const f32x2 ww = pk(w, w);
            llo = fma2(ww, add2(zlo, xlo), llo);
            lhi = fma2(ww, add2(zhi, xhi), lhi);
        }
        const f32x2 k2lo = pk(k2[0], k2[1]), k2hi = pk(k2[2], k2[3]);
        const f32x2 dulo = pk(du[0], du[1]), duhi = pk(du[2], du[3]);
        f32x2 dlo, dhi;
        if (sxc == 0.f && !zdamp) {
            dlo = fma2(k2lo, llo, dulo);          // K1 = 1 exactly
            dhi = fma2(k2hi, lhi, duhi);
        } else {
            float k1[4];
#pragma unroll
            for (int e = 0; e < 4; e++) k1[e] = sxc == 0.f ? k1z[e] : (dzv[e] == 0.f ? k1xc : k1_of(sxc + dzv[e]));
            dlo = fma2(pk(k1[0], k1[1]), dulo, mul2(k2lo, llo));
            dhi = fma2(pk(k1[2], k1[3]), duhi, mul2(k2hi, lhi));
        }
        if (imask & (1u << rr)) {   // a3: K2 * scale * w * val
            const float4 iv = injs[rr * 128 + tid];
            dlo = fma2(k2lo, pk(iv.x, iv.y), dlo);
            dhi = fma2(k2hi, pk(iv.z, iv.w), dhi);
        }
        const f32x2 ulo = add2(clo, dlo), uhi = add2(chi, dhi);
        float4 dn, un;
        upk(dlo, dn.x, dn.y); upk(dhi, dn.z, dn.w);
        upk(ulo, un.x, un.y); upk(uhi, un.z, un.w);
        if (!full) {   // ragged quad at the end of a row: keep the halo zero
            if (jz + 1 >= L.Pz) { dn.y = 0.f; un.y = 0.f; }
            if (jz + 2 >= L.Pz) { dn.z = 0.f; un.z = 0.f; }
            dn.w = 0.f; un.w = 0.f;
        }
        st4(d0 + off, dn);
        st4(n0 + off, un);
        const int ix = jx - L.nb;
        if (zphys && ix >= 0 && ix < L.nx) stcs4(a.hist + (long long)ix * L.upz + iz, un);
    }
    }   // active
    DBG_STAMP(a, 6);
}

}  // namespace rtm
