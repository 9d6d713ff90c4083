// acoustic2d_resident.cuh -- 2D isotropic acoustic time stepping (a1) with the wavefield RESIDENT IN SHARED MEMORY for a
// whole time block of up to T steps: one cooperative launch per time block instead of one launch per step.
//
// Why.  At c1 (1911 x 911 padded points) one step through L2 moves ~60 MB (u, du, K2 in, u', du', history out, plus the
// flush role's planes): about 5 us at the L2 slice throughput, behind a grid-wide dependency per step (9.8 us measured
// for acoustic2d_stream_kernel).  But u (two time levels) and du of the whole grid are 21 MB and the 148 SMs hold 33 MB
// of shared memory: the fields need not leave the chip at all.
//
// How.  The padded grid is cut along x into NB slabs of R or R+1 consecutive rows, one block (= one SM) per slab.  A block
// keeps u_old / u_new of its rows plus a halo of 4 rows on either side, and du of its rows, in shared memory.  One step:
//   1. sweep: thread = one z-quad column of a row group, streaming along x with the 9-deep register queue of the
//      streaming kernel (same operations in the same order per point: the results are bit-identical to it); K2 comes
//      from L2 (read-only, 4 B / point / step), everything else from shared memory; fused damping, injection (a3, amounts
//      staged per (row, quad) group), history store of the probed field (a5, the only DRAM stream of the kernel);
//   2. publish: the first and the last 4 rows of u_new go to a double-buffered exchange buffer in global memory (L2);
//      one thread releases the block's step counter (fence + store; the pattern of a split-phase grid barrier, but
//      between NEIGHBOURS only: a block never waits for more than the two blocks it exchanges rows with);
//   3. acquire the two neighbours' counters, copy their 4 + 4 rows into the halo rows of u_new;
//   4. deferred-free receiver sampling (a4) of the rows the block owns (bilinear corners reach at most one row into the
//      halo), straight from shared memory.
// The launch is cooperative (all NB <= #SM blocks are co-resident by construction), spins are bounded (a protocol bug
// ends in a trap, not in a hung GPU).  At the end of the launch u and du go back to global memory, so everything around
// the time loop (snapshots, the flush of the history ring into the probe planes, the next launch) sees the usual arrays.
#pragma once
#include "common.cuh"

namespace rtm {

constexpr int RS_THREADS = 512;
constexpr int RS_MAXG = 255;      // injection groups (row, quad) per block (index + 1 fits a byte)
constexpr int RS_MAXS = 256;      // sampled points per block
constexpr int RS_MAXROWS = 64;    // rows per slab the tables are sized for
constexpr int RS_MAXE = 256;      // injection entries per block (cached in shared memory)

struct ResidentArgs {
    int NB;                 // blocks = slabs
    int rbase, rrem;        // slab b owns rbase + (b < rrem) rows, starting at b * rbase + min(b, rrem)
    int rmax;               // rbase + (rrem > 0)
    int nq;                 // z-quads per row = ceil(Pz / 4)
    int spz;                // floats per shared-memory row of u: [4 zeros | 4 nq | 4 zeros]
    int groups;             // row groups per slab (threads = nq * groups tasks)
    int nsteps;             // steps in this launch
    int n0, dir;            // time index of the first step, +1 forward / -1 adjoint
    int ninj;               // columns of a value row
    const float *inj_base;  // [nt][ninj]
    float *smp_base;        // [nt][nsmp] or NULL
    float *hist0;           // history slot of the first step of the launch (NULL: no probing)
    float *u, *du;          // the field arrays in global memory (cur; read at the start, written at the end)
    float *xbuf;            // exchange buffer [2][NB][2][4][4 nq]
    unsigned *flags;        // step counters, one per block, 32 words apart
    unsigned ep0;           // counter value before the first step of this launch
    int *err;               // set to 1 before a trap (diagnostics)
};

__device__ __forceinline__ unsigned ld_acquire(const unsigned *p) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(unsigned *p, unsigned v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// store into the shared memory of block `rank` of the cluster, at the address that `p` has in this block
__device__ __forceinline__ void st_cluster4(float *p, int rank, float4 v) {
    unsigned remote;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(remote) : "r"(smem_u32(p)), "r"(rank));
    asm volatile("st.shared::cluster.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(remote), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}
__device__ __forceinline__ float4 ldcg4(const float *p) { return __ldcg(reinterpret_cast<const float4 *>(p)); }

#ifdef RTM_DEBUG
#define RS_STAMP(slot) do { if ((a.dbg & 16) && (tid == 0 || tid == RS_THREADS - 32) && s == ra.nsteps - 1) a.dbg_ts[b * 8 + (slot)] = gtimer(); } while (0)
#else
#define RS_STAMP(slot) do { } while (0)
#endif

struct RsGroup { int e0, e1; short row, col; };          // injection entries [e0, e1) feed quad `col` of local row `row`
struct RsSample { int o[4]; float w[4]; int j; };        // shared-memory offsets of the corners, weights, output column

// CL = true: all slabs form ONE thread-block cluster (<= 16 blocks): boundary rows go straight into the neighbours'
// halo rows through distributed shared memory and a step ends with a cluster barrier -- no exchange buffer, no
// counters, no communication warp; every thread takes a short run of rows (down to one), because a grid this small is
// bound by latency, not by work.  CL = false: slabs exchange through L2 as described above.
template <bool CL>
__global__ void __launch_bounds__(RS_THREADS, 1) acoustic2d_resident_kernel(const __grid_constant__ StepArgs a,
                                                                         const __grid_constant__ ResidentArgs ra) {
    extern __shared__ __align__(16) float rs_smem[];
    const Layout &L = a.L;
    const int tid = threadIdx.x, b = blockIdx.x;
    const int R = ra.rbase + (b < ra.rrem ? 1 : 0);
    const int r0 = b * ra.rbase + min(b, ra.rrem);          // first padded row of the slab
    const int nq = ra.nq, spz = ra.spz, nq4 = nq * 4;
    const int urows = ra.rmax + 8;

    // ---- shared memory carve --------------------------------------------------------------------------------------
    float *U0 = rs_smem;                                   // [urows][spz]
    float *U1 = U0 + urows * spz;
    float *D = U1 + urows * spz;                           // [rmax][nq4]
    float *Ks = D + ra.rmax * nq4;                         // CL only: K2 of the slab [rmax][nq4] (a small grid has the room)
    float4 *staged = reinterpret_cast<float4 *>(Ks + (CL ? ra.rmax * nq4 : 0));   // [RS_MAXG + 1]: this step's injection amounts
    InjEntry *ecache = reinterpret_cast<InjEntry *>(staged + RS_MAXG + 1);   // [RS_MAXE]: the slab's injection entries
    float *vbuf = reinterpret_cast<float *>(ecache + RS_MAXE);              // [2][RS_MAXE]: their values for this / the next step (cp.async)
    RsGroup *grp = reinterpret_cast<RsGroup *>(vbuf + 2 * RS_MAXE);          // [RS_MAXG]
    RsSample *smp = reinterpret_cast<RsSample *>(grp + RS_MAXG + 1);          // [RS_MAXS]
    unsigned char *gmap = reinterpret_cast<unsigned char *>(smp + RS_MAXS);   // [rmax][nq]: group index + 1
    __shared__ int s_ngrp, s_nsmp;
    __shared__ int s_rowg[RS_MAXROWS + 1];                 // first group of every local row
    __shared__ float s_dx[RS_MAXROWS + 1], s_k1x[RS_MAXROWS + 1];
    __shared__ __align__(8) unsigned long long s_hbar;     // mbarrier of the halo rows (one phase per step)

    // ---- launch prologue ------------------------------------------------------------------------------------------
    for (int i = tid; i < 2 * urows * spz; i += RS_THREADS) U0[i] = 0.f;       // halo rows / pad columns of the edge slabs stay 0
    for (int i = tid; i < ra.rmax * nq; i += RS_THREADS) gmap[i] = 0;
    if (tid == 0) { s_ngrp = 0; s_nsmp = 0; }
    __syncthreads();
    // u: own rows and the halo rows that exist; du: own rows
    for (int i = tid; i < (R + 8) * nq; i += RS_THREADS) {
        const int lr = i / nq, col = i - lr * nq;
        const int jx = r0 - 4 + lr;
        if (jx >= 0 && jx < L.Px) st4(U0 + lr * spz + 4 + col * 4, ld4(ra.u + L.org + (long long)jx * L.sx + col * 4));
    }
    for (int i = tid; i < R * nq; i += RS_THREADS) {
        const int lr = i / nq, col = i - lr * nq;
        st4(D + lr * nq4 + col * 4, ld4(ra.du + L.org + (long long)(r0 + lr) * L.sx + col * 4));
    }
    if (CL)
        for (int i = tid; i < R * nq; i += RS_THREADS) {
            const int lr = i / nq, col = i - lr * nq;
            st4(Ks + lr * nq4 + col * 4, ld4(a.K2 + L.org + (long long)(r0 + lr) * L.sx + col * 4));
        }
    const int ebase = a.row_start[r0], nent_b = min(a.row_start[r0 + R] - ebase, RS_MAXE);   // the host checked the cap
    for (int i = tid; i < nent_b; i += RS_THREADS) ecache[i] = a.ent[ebase + i];
    // injection groups: the entries of a row are sorted by jz, so the entries of one quad are contiguous; one thread
    // per row counts its groups, a serial prefix over <= RS_MAXROWS rows places them (deterministic order)
    if (tid < R) {
        const int e0 = a.row_start[r0 + tid], e1 = a.row_start[r0 + tid + 1];
        int n = 0, last = -1;
        for (int e = e0; e < e1; e++) { const int c = a.ent[e].jz >> 2; if (c != last) { n++; last = c; } }
        s_rowg[tid + 1] = n;
    }
    __syncthreads();
    if (tid == 0) {
        s_rowg[0] = 0;
        for (int i = 0; i < R; i++) s_rowg[i + 1] += s_rowg[i];
        s_ngrp = s_rowg[R];
    }
    __syncthreads();
    if (tid < R) {
        const int e0 = a.row_start[r0 + tid], e1 = a.row_start[r0 + tid + 1];
        int g = s_rowg[tid] - 1, last = -1;
        for (int e = e0; e < e1; e++) {
            const int c = a.ent[e].jz >> 2;
            if (c != last) {
                g++; last = c;
                if (g < RS_MAXG) { grp[g].e0 = e; grp[g].row = (short)tid; grp[g].col = (short)c; gmap[tid * nq + c] = (unsigned char)(g + 1); }
            }
            if (g < RS_MAXG) grp[g].e1 = e + 1;
        }
    }
    // sampled points whose first corner lies in the slab (the other corners reach at most one row further: halo)
    if (ra.smp_base != nullptr) {
        for (int j = tid; j < a.nsmp; j += RS_THREADS) {
            const int i0 = a.smp_idx[4 * (size_t)j] - (int)L.org;
            const int jx = i0 / (int)L.sx;
            if (jx >= r0 && jx < r0 + R) {
                const int k = atomicAdd(&s_nsmp, 1);
                if (k < RS_MAXS) {
                    RsSample s;
                    s.j = j;
                    for (int c = 0; c < 4; c++) {
                        const int ii = a.smp_idx[4 * (size_t)j + c] - (int)L.org;
                        const int cx = ii / (int)L.sx, cz = ii - cx * (int)L.sx;
                        s.w[c] = a.smp_w[4 * (size_t)j + c];
                        s.o[c] = s.w[c] != 0.f ? (cx - r0 + 4) * spz + 4 + cz : 0;
                    }
                    smp[k] = s;
                }
            }
        }
    }
    __syncthreads();
    const int ngrp = min(s_ngrp, RS_MAXG), nsmp_b = min(s_nsmp, RS_MAXS);   // the host checked the caps (rtm.cu: build_geometry)
    if (CL) {   // no block writes into a neighbour's shared memory before that neighbour has set it up
        asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
        asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
    }

    // ---- roles ---------------------------------------------------------------------------------------------------------
    // Warps 0 .. 14 sweep: thread = z-quad column `col`, streaming from an EDGE of the slab towards its middle -- group 0
    // downwards from row 0, group 1 upwards from row R-1 -- so that the 4 + 4 rows the neighbours need are computed (and
    // published) first and the interior rows overlap the exchange.  Warp 15 is the communication warp: it releases the
    // slab's step counter once every sweeping thread has published its boundary rows (named barrier 1), acquires the
    // neighbours' counters and asks the copy engine for their 4 + 4 rows (cp.async.bulk -> halo rows of u_new, counted
    // on an mbarrier).  Streaming upwards uses the same expressions with the two x neighbours of a pair swapped;
    // IEEE addition commutes, so the bits do not depend on the direction.
    constexpr int RS_SWEEP = RS_THREADS - 32;
    const bool comm = !CL && tid >= RS_SWEEP;
    const int ngroups = CL ? ra.groups : 2;           // CL: `groups` row groups, all streaming downwards
    const bool has_task = tid < ngroups * nq;         // the host makes groups * nq <= RS_SWEEP
    const int tg = has_task ? tid / nq : 0, col = has_task ? tid - tg * nq : 0;
    const int mid = (R + 1) / 2;                      // !CL: group 0: rows 0 .. mid-1; group 1: rows R-1 .. mid
    const int glo = (int)((long long)R * tg / ngroups), ghi = (int)((long long)R * (tg + 1) / ngroups);
    const int nrow_t = !has_task ? 0 : CL ? ghi - glo : (tg == 0 ? mid : R - mid);
    const int rstart = CL ? glo : (tg == 0 ? 0 : R - 1), dirn = (CL || tg == 0) ? 1 : -1;
    const int nbnd = (CL || R < 8) ? nrow_t : min(nrow_t, 4);   // leading rows of the stream that may feed a neighbour
    const int jz = col * 4;
    float dzv[4] = {0.f, 0.f, 0.f, 0.f}, k1z[4] = {1.f, 1.f, 1.f, 1.f};
    if (has_task) {
        const float4 d4 = ld4(a.dampz + jz), k4 = ld4(a.k1z + jz);
        dzv[0] = d4.x; dzv[1] = d4.y; dzv[2] = d4.z; dzv[3] = d4.w;
        k1z[0] = k4.x; k1z[1] = k4.y; k1z[2] = k4.z; k1z[3] = k4.w;
    }
    const bool zdamp = (dzv[0] != 0.f) | (dzv[1] != 0.f) | (dzv[2] != 0.f) | (dzv[3] != 0.f);
    const bool full = jz + 3 < L.Pz;
    const int iz = jz - L.nbz;
    const bool zphys = has_task && iz >= 0 && iz < L.nz && ra.hist0 != nullptr;
    unsigned imask = 0;                           // bit i: the i-th row of this thread's stream has an injection group (<= 32 rows)
    for (int i = 0; i < nrow_t; i++)
        if (gmap[(rstart + i * dirn) * nq + col]) imask |= 1u << i;
    // x damping tables of the slab's rows in shared memory (the L1 that is left beside 200+ KB of shared memory does
    // not keep them: a load per row from L2 sat on the critical path of every row)
    for (int i = tid; i < R; i += RS_THREADS) { s_dx[i] = a.dampx[r0 + i]; s_k1x[i] = a.k1x[r0 + i]; }
    if (tid == 0) { mbar_init(&s_hbar, 1); mbar_fence_init(); }
    __syncthreads();
    const long long ksx = (long long)dirn * L.sx;
    const float *K2p = a.K2 + L.org + (long long)(r0 + rstart) * L.sx + jz;     // K2 of the first row of the stream
    const int rs = dirn * spz, rs4 = 4 * rs;                                       // shared-memory row stride of the stream
    const int dstep = dirn * nq4;
    const long long hstep = (long long)dirn * L.upz;

    float *Uo = U0, *Un = U1;
    unsigned *my_flag = ra.flags + 32 * b;
    const unsigned *lf = b > 0 ? ra.flags + 32 * (b - 1) : nullptr, *rf = b + 1 < ra.NB ? ra.flags + 32 * (b + 1) : nullptr;
    const unsigned hbytes = (unsigned)((lf ? 4 : 0) + (rf ? 4 : 0)) * (unsigned)nq4 * 4u;

    // The values of the slab's injection entries for step n travel by cp.async (4 bytes each) into vbuf[buf] while the
    // previous step is swept; stage() then forms the amounts v = sum_i scale w_i val_i per lane of each (row, quad) group,
    // in entry order (C27), from shared memory only: nothing on the critical path of a step waits for L2.
    auto fetch_values = [&](int n, int buf) {
        const float *val = ra.inj_base + (size_t)n * ra.ninj;
        for (int e = tid; e < nent_b; e += RS_THREADS) {
            const unsigned dsts = smem_u32(vbuf + buf * RS_MAXE + e);
            asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dsts), "l"(val + ecache[e].id) : "memory");
        }
        cp_async_commit();
    };
    auto stage = [&](int buf) {
        if (tid < ngrp) {
            const RsGroup g = grp[tid];
            float acc[4] = {0.f, 0.f, 0.f, 0.f};
            for (int e = g.e0 - ebase; e < g.e1 - ebase; e++) {
                const InjEntry en = ecache[e];
                const int dz = en.jz - 4 * g.col;
                const float v = a.inj_scale * en.w * vbuf[buf * RS_MAXE + e];
#pragma unroll
                for (int q = 0; q < 4; q++)
                    if (q == dz) acc[q] += v;
            }
            staged[tid] = make_float4(acc[0], acc[1], acc[2], acc[3]);
        }
    };
    fetch_values(ra.n0, 0);
    cp_async_wait<0>();
    __syncthreads();

    for (int s = 0; s < ra.nsteps; s++) {
        const int n = ra.n0 + s * ra.dir;
        const unsigned ep = ra.ep0 + (unsigned)s + 1u;
        float *xb = ra.xbuf + ((size_t)(ep & 1u) * ra.NB + b) * (size_t)(8 * nq4);
        RS_STAMP(0);
        stage(s & 1);                                      // this step's amounts (values fetched during the previous step)
        if (s + 1 < ra.nsteps) fetch_values(n + ra.dir, (s + 1) & 1);
        __syncthreads();
        if (!comm) {
            // ---- sweep: boundary rows first, then towards the middle ----------------------------------------------
            {
                // running pointers of the stream (one add per row each: no index arithmetic inside the row)
                const float *up = Uo + (rstart + 4) * spz + 4 + jz;     // u_old, this column, current row
                float *unp = Un + (rstart + 4) * spz + 4 + jz;          // u_new
                float *dp = D + rstart * nq4 + jz;                      // du
                const float *kp = K2p + 2 * ksx;                        // K2 two rows ahead
                float *hp = ra.hist0 + (long long)s * a.pNu + (long long)(r0 + rstart - L.nb) * L.upz + iz;   // dereferenced on physical rows only
                float *xp = xb + (tg == 0 ? 0 : 7) * nq4 + jz;          // exchange row of the stream's first row (valid while rr is a boundary row)
                int rr = rstart;
                unsigned im = imask;
                float4 q[9];                                            // stream rows i-4 .. i+4
#pragma unroll
                for (int i = 0; i < 8; i++) q[i] = (nrow_t > 0 ? ld4(up + (i - 4) * rs) : make_float4(0.f, 0.f, 0.f, 0.f));
                const float *ksp = Ks + rstart * nq4 + jz;              // CL: K2 of the current row in shared memory
                float4 k24 = make_float4(0.f, 0.f, 0.f, 0.f), k24n = k24;
                if (!CL) { k24 = nrow_t > 0 ? ldg4(K2p) : k24; k24n = nrow_t > 1 ? ldg4(K2p + ksx) : k24; }
                auto row = [&](int i, bool publish) {
                    q[8] = ld4(up + rs4);
                    const float4 c = q[4];
                    const float4 zm = ld4(up - 4), zp = ld4(up + 4);
                    const float4 du4 = ld4(dp);
                    const float4 k2c = CL ? ld4(ksp) : k24;
                    if (!CL) {
                        k24 = k24n;
                        if (i + 2 < nrow_t) k24n = ldg4(kp);   // K2 (L2) two rows ahead of its use
                    }
                    const float sxc = s_dx[rr], k1xc = s_k1x[rr];
                    const float win[12] = {zm.x, zm.y, zm.z, zm.w, c.x, c.y, c.z, c.w, zp.x, zp.y, zp.z, zp.w};
                    const float cc[4] = {c.x, c.y, c.z, c.w};
                    // the same operations in the same order per point as acoustic2d_stream_kernel
                    const f32x2 clo = pk(c.x, c.y), chi = pk(c.z, c.w);
                    f32x2 llo = pk(0.f, 0.f), lhi = llo;
#pragma unroll
                    for (int j = 4; j >= 1; j--) {
                        const float4 P = q[4 + j], M = q[4 - j];
                        const f32x2 xlo = dd2(pk(P.x, P.y), pk(M.x, M.y), clo), xhi = dd2(pk(P.z, P.w), pk(M.z, M.w), chi);
                        f32x2 zlo, zhi;
                        if (j % 2 == 0) {
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
                    const f32x2 k2lo = pk(k2c.x, k2c.y), k2hi = pk(k2c.z, k2c.w);
                    const f32x2 dulo = pk(du4.x, du4.y), duhi = pk(du4.z, du4.w);
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
                    if (im & 1u) {   // a3: K2 * scale * w * val
                        const float4 iv = staged[gmap[rr * nq + col] - 1];
                        dlo = fma2(k2lo, pk(iv.x, iv.y), dlo);
                        dhi = fma2(k2hi, pk(iv.z, iv.w), dhi);
                    }
                    im >>= 1;
                    const f32x2 ulo = add2(clo, dlo), uhi = add2(chi, dhi);
                    float4 dn, un;
                    upk(dlo, dn.x, dn.y); upk(dhi, dn.z, dn.w);
                    upk(ulo, un.x, un.y); upk(uhi, un.z, un.w);
                    if (!full) {   // ragged quad at the end of a row: keep the halo zero
                        if (jz + 1 >= L.Pz) { dn.y = 0.f; un.y = 0.f; }
                        if (jz + 2 >= L.Pz) { dn.z = 0.f; un.z = 0.f; }
                        dn.w = 0.f; un.w = 0.f;
                    }
                    st4(dp, dn);
                    st4(unp, un);
                    if (zphys && (unsigned)(r0 + rr - L.nb) < (unsigned)L.nx) stcs4(hp, un);
                    if (publish) {
                        // the first 4 rows of the slab feed the left neighbour, the last 4 the right one (a slab of fewer
                        // than 8 rows has rows that feed both)
                        if (CL) {
                            // straight into the neighbour's halo rows (same shared-memory layout, same u_new buffer)
                            // my row rr (shared-memory row rr + 4) is the left neighbour's row R_left + 4 + rr and the right
                            // neighbour's row rr - (R - 4)
                            if (rr < 4 && b > 0) st_cluster4(unp + (ra.rbase + (b - 1 < ra.rrem ? 1 : 0)) * spz, b - 1, un);
                            if (rr >= R - 4 && b + 1 < ra.NB) st_cluster4(unp - R * spz, b + 1, un);
                        } else {
                            if (rr < 4) __stcg(reinterpret_cast<float4 *>(xb + rr * nq4 + jz), un);
                            if (rr >= R - 4) __stcg(reinterpret_cast<float4 *>(xb + (4 + rr - (R - 4)) * nq4 + jz), un);
                        }
                    }
                    up += rs; unp += rs; dp += dstep; kp += ksx; ksp += dstep; hp += hstep; rr += dirn;
#pragma unroll
                    for (int k = 0; k < 8; k++) q[k] = q[k + 1];
                };
                (void)xp;
                // boundary rows; then every warp arrives as a whole (the rows its neighbours need are published); then the
                // interior rows, which overlap the exchange
#pragma unroll 1
                for (int i = 0; i < nbnd; i++) row(i, true);
                if (!CL) {
                    __syncwarp();
                    asm volatile("bar.arrive 1, %0;" ::"n"(RS_THREADS) : "memory");
                }
#pragma unroll 1
                for (int i = nbnd; i < nrow_t; i++) row(i, false);
            }
            RS_STAMP(1);
        } else {
            // ---- communication warp ---------------------------------------------------------------------------------
            asm volatile("bar.sync 1, %0;" ::"n"(RS_THREADS) : "memory");      // every boundary row of the slab is published
            if (tid == RS_SWEEP) {
                st_release(my_flag, ep);        // fence.acq_rel.gpu + store: cumulative over the block's stores before the barrier
                if (hbytes) mbar_arrive_expect_tx(&s_hbar, hbytes);
                for (int side = 0; side < 2; side++) {
                    const unsigned *f = side == 0 ? lf : rf;
                    if (f == nullptr) continue;
                    int it = 0;
                    while ((int)(ld_acquire(f) - ep) < 0)
                        if (++it > (1 << 24)) { *ra.err = 1; __threadfence_system(); __trap(); }
                    asm volatile("fence.proxy.async;" ::: "memory");
                    // left neighbour's LAST 4 rows -> halo rows 0..3; right neighbour's FIRST 4 rows -> rows R+4..R+7
                    const int nbk = side == 0 ? b - 1 : b + 1;
                    const float *src = ra.xbuf + ((size_t)(ep & 1u) * ra.NB + nbk) * (size_t)(8 * nq4) + (side == 0 ? 4 : 0) * nq4;
                    for (int k = 0; k < 4; k++) {
                        float *dst = Un + ((side == 0 ? k : R + 4 + k) * spz + 4);
                        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                                     ::"r"(smem_u32(dst)), "l"(src + k * nq4), "r"((unsigned)nq4 * 4u), "r"(smem_u32(&s_hbar)) : "memory");
                    }
                }
            }
            RS_STAMP(2);
        }
        cp_async_wait<0>();                                    // this thread's share of the next step's values has landed
        if (CL) {
            // every block of the cluster has written its rows (and its neighbours' halo rows): release / acquire at cluster scope
            asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
            asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
        } else {
            __syncthreads();                                   // u_new of the slab is complete, next amounts staged
            RS_STAMP(3);
            if (hbytes) mbar_wait(&s_hbar, (unsigned)s & 1u);  // ... and the neighbours' rows have landed in its halo rows
        }
        RS_STAMP(4);
        // ---- receiver sampling of this step's field (a4) ----------------------------------------------------------------
        if (tid < nsmp_b) {
            const RsSample sp = smp[tid];
            float acc = 0.0f;
#pragma unroll
            for (int c = 0; c < 4; c++)
                if (sp.w[c] != 0.0f) acc = fmaf(sp.w[c], Un[sp.o[c]], acc);
            ra.smp_base[(size_t)n * a.nsmp + sp.j] = a.smp_scale * acc;
        }
        RS_STAMP(6);
        float *t = Uo; Uo = Un; Un = t;
    }
    // ---- back to global memory --------------------------------------------------------------------------------------
    __syncthreads();
    for (int i = tid; i < R * nq; i += RS_THREADS) {
        const int lr = i / nq, cq = i - lr * nq;
        const long long o = L.org + (long long)(r0 + lr) * L.sx + cq * 4;
        st4(ra.u + o, ld4(Uo + (lr + 4) * spz + 4 + cq * 4));
        st4(ra.du + o, ld4(D + lr * nq4 + cq * 4));
    }
}

}  // namespace rtm
