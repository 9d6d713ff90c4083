// common.cuh -- layouts, argument blocks and small device helpers shared by the kernels.
// (CUDA path only; nothing here is used by oracle/.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace rtm {

// Internal HBM layout.
//  Fields / coefficient arrays: padded grid P plus a zero halo of H points on every side of every
//  active axis, z contiguous with pitch pz (multiple of 32 floats); point (jx,jy,jz) of P lives at
//  org + jx*sx + jy*sy + jz.  H = 4 (acoustic, order-8 star) or 8 (TTI, two chained order-8 first
//  derivatives).  org, sx, sy are multiples of 4 floats so that z-quads (jz % 4 == 0) are float4-aligned.
//  Compressed wavefields Uz/Vz: [k][ix][iy][iz] on the PHYSICAL grid only (reading C12), z pitch upz
//  (multiple of 32), plane stride Nu.  The internal z axis starts zs points before the padded grid so that the
//  physical grid starts at a multiple of 4 (nbz): physical and padded quads are aligned for any nb.  Those zs
//  points have K2 = 0 (and cos = sin = 0), so every field stays exactly zero there, like the halo.
struct Layout {
    int nd;
    int nx, ny, nz;
    int Px, Py, Pz;   // Pz is the INTERNAL z extent: zs alignment points (K2 = 0: they stay zero) + the padded grid
    int Pzc, zs;      // canonical padded z extent nz + 2 nb; zs = (4 - nb % 4) % 4 makes nbz a multiple of 4
    int nb, nby;      // nby = nb in 3D, 0 in 2D (the dummy y axis has no layer)
    int nbz;          // internal z index of the first physical point = nb + zs
    int H, Hy;     // Hy = H in 3D, 0 in 2D
    int pz;
    long long sx, sy;
    long long org;
    long long fsize;   // floats per field (incl. slack)
    int upz;
    long long Nu;      // floats per probe plane
};

struct InjEntry {
    int jz;    // padded z index of the grid point
    int id;    // source / receiver index (column of the value row)
    float w;   // multilinear corner weight
    int pad;
};

// One time step (acoustic: one field; TTI: p and r).
struct StepArgs {
    Layout L;
    const float *u0, *u1;   // current field(s)   (u1: TTI r)
    float *n0, *n1;         // new field(s)
    float *d0, *d1;         // increment(s) du = u_cur - u_prev, updated in place
    const float *K2, *epsh, *delh, *cs, *sn;
    const float *cp, *sp;   // 3D TTI: cos / sin of the azimuth (cs, sn: of the tilt)
    float *F[6];            // 3D TTI: the six intermediate vector components (tti3d.cuh)
    const float *dampx, *dampy, *dampz;
    const float *k1x, *k1y, *k1z;   // per-axis K1 tables: k1a[j] = (1 - damp_a[j]) / (1 + damp_a[j])
    int adjoint;
#ifdef RTM_DEBUG
    int dbg;
    unsigned long long *dbg_ts;   // timing experiments (dbg & 16): per-phase %globaltimer stamps, [block][8]
#endif
    // 3D streaming kernel: four CUtensorMaps (128 B each) in device memory: u ping, u pong, K2, du (rtm.cu: make_tmaps)
    const void *tmaps;
    int tm_u;               // which of the two u maps describes u0 in this launch
    // fused probe: PZ[k][x] += Zrow[k] * new[x]
    float *PZ;
    const float *Zrow;
    int r;
    int two;                // TTI, probe_fields = 2 (reading C29): plane 2k of PZ = probe k of p, plane 2k + 1 = probe k of r
    long long pNu;          // floats per probe-plane group and per history slot: Nu, or 2 Nu with two probed fields (the
                            // r field then sits Nu floats behind the p field: to the flush roles it is nx more rows)
    // time-blocked probing: instead of PZ, store the probed field into this history slot (physical grid,
    // probe-plane layout); probe_flush_kernel applies T rows of Z at once
    float *hist;
    // ... and the leading fl_blocks blocks of every step launch flush one slice (pairs [fl_q0, fl_q1) of
    // float2 units of the physical grid) of the PREVIOUS time block's history into PZ, so that the
    // DRAM-bound probe update overlaps the L2/latency-bound stencil inside one launch
    const float *fl_hist;   // slot 0 of the time block being flushed
    const float *fl_Z0;     // Z row of that block's slot 0
    long long fl_zstep;     // +zr forward, -zr adjoint
    int fl_n;               // slots in that block
    int fl_blocks;
    int fl_nowait;          // the flush role may skip griddepcontrol.wait (its inputs are >= 2 launches old)
    long long fl_q0, fl_q1;   // slice of this launch in units of float2 (flush_role) or float4 (flush_role4)
    int zr;
    unsigned gx, gy;        // stencil grid extents (the launch grid is 1-D: fl_blocks + gx*gy*gz)
    // fused injection (row-CSR over (jx,jy) rows, restricted to a bounding box)
    const int *row_start;
    const InjEntry *ent;
    const float *inj_val;   // value row of this step [ninj]
    float inj_scale;
    int bx0, bx1, by0, by1, bz0, bz1;
    // deferred sampling of the CURRENT field (= previous step's result) into smp_out[nsmp]
    const int *smp_idx;     // [nsmp][nc] offsets from the field base
    const float *smp_w;     // [nsmp][nc]
    float *smp_out;         // NULL: nothing to sample in this launch
    int nsmp, nc;
    float smp_scale;
};

// order-8 weights (textbook Fornberg), as the fp32 constants both sides round to (reading C18)
__device__ __forceinline__ float w2(int j) {
    return j == 1 ? (float)(8.0 / 5.0) : j == 2 ? (float)(-1.0 / 5.0) : j == 3 ? (float)(8.0 / 315.0) : (float)(-1.0 / 560.0);
}
__device__ __forceinline__ float w1(int j) {
    return j == 1 ? (float)(4.0 / 5.0) : j == 2 ? (float)(-1.0 / 5.0) : j == 3 ? (float)(4.0 / 105.0) : (float)(-1.0 / 280.0);
}

__device__ __forceinline__ float4 ld4(const float *p) { return *reinterpret_cast<const float4 *>(p); }
__device__ __forceinline__ float4 ldg4(const float *p) { return __ldg(reinterpret_cast<const float4 *>(p)); }
__device__ __forceinline__ void st4(float *p, float4 v) { *reinterpret_cast<float4 *>(p) = v; }
// streaming (evict-first) accesses for the probe planes: read once + written once per step
__device__ __forceinline__ float4 ldcs4(const float *p) { return __ldcs(reinterpret_cast<const float4 *>(p)); }
__device__ __forceinline__ void stcs4(float *p, float4 v) { __stcs(reinterpret_cast<float4 *>(p), v); }

// Packed fp32x2 arithmetic (sm_100: FADD2 / FMUL2 / FFMA2, one issue slot for two IEEE-rn fp32 operations).  A pair
// is carried in a 64-bit register; pk/upk compile to nothing when the two floats sit in an aligned register pair
// (the halves of a float4 do).  Each lane rounds exactly like the scalar instruction, so results are unchanged.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk(float a, float b) { f32x2 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void upk(f32x2 p, float &a, float &b) { asm("mov.b64 {%0,%1}, %2;" : "=f"(a), "=f"(b) : "l"(p)); }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) { f32x2 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) { f32x2 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) { f32x2 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
// (P - c) + (M - c) on a pair: the "difference form" term of the Laplacian (reading C21)
__device__ __forceinline__ f32x2 dd2(f32x2 P, f32x2 M, f32x2 c) { return add2(sub2(P, c), sub2(M, c)); }

// The same pair interface with a compile-time switch between the packed instructions and two scalar ones
// (A/B timing of FADD2 / FFMA2 against FADD / FFMA; both give identical bits).
template <bool PK> struct V2;
template <> struct V2<true> {
    typedef f32x2 T;
    static __device__ __forceinline__ T mk(float a, float b) { return pk(a, b); }
    static __device__ __forceinline__ void get(T p, float &a, float &b) { upk(p, a, b); }
    static __device__ __forceinline__ T add(T a, T b) { return add2(a, b); }
    static __device__ __forceinline__ T sub(T a, T b) { return sub2(a, b); }
    static __device__ __forceinline__ T mul(T a, T b) { return mul2(a, b); }
    static __device__ __forceinline__ T fma(T a, T b, T c) { return fma2(a, b, c); }
    static __device__ __forceinline__ T dd(T P, T M, T c) { return dd2(P, M, c); }
};
template <> struct V2<false> {
    typedef float2 T;
    static __device__ __forceinline__ T mk(float a, float b) { return make_float2(a, b); }
    static __device__ __forceinline__ void get(T p, float &a, float &b) { a = p.x; b = p.y; }
    static __device__ __forceinline__ T add(T a, T b) { return make_float2(a.x + b.x, a.y + b.y); }
    static __device__ __forceinline__ T sub(T a, T b) { return make_float2(a.x - b.x, a.y - b.y); }
    static __device__ __forceinline__ T mul(T a, T b) { return make_float2(a.x * b.x, a.y * b.y); }
    static __device__ __forceinline__ T fma(T a, T b, T c) { return make_float2(fmaf(a.x, b.x, c.x), fmaf(a.y, b.y, c.y)); }
    static __device__ __forceinline__ T dd(T P, T M, T c) { return add(sub(P, c), sub(M, c)); }
};

// 16-byte asynchronous copy global -> shared; ok == false writes zeros (the source is not read)
__device__ __forceinline__ void cp_async16(float *dst_smem, const float *src, bool ok) {
    const unsigned d = (unsigned)__cvta_generic_to_shared(dst_smem);
    const int n = ok ? 16 : 0;
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(src), "r"(n) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// ---- TMA (cp.async.bulk.tensor) + mbarrier: one elected thread asks the copy engine for a whole box of a tensor
// described by a CUtensorMap; the bytes land in shared memory and are counted on an mbarrier the consumers wait on.
// (SASS: UTMALDG / SYNCS.)  Out-of-bounds parts of a box are filled with zeros.
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
// one arrival that also announces `bytes` of copy-engine traffic for the current phase
__device__ __forceinline__ void mbar_arrive_expect_tx(unsigned long long *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// Wait for the phase with the given parity.  try_wait sleeps in hardware for a bounded time; the retry count is bounded
// too, so a descriptor or byte-count bug ends in a trap (a CUDA error on the host), never in a hung GPU.
__device__ __forceinline__ void mbar_wait(unsigned long long *bar, unsigned parity) {
    const unsigned a = smem_u32(bar);
    unsigned done = 0;
    for (int it = 0; it < (1 << 22); it++) {
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(done) : "r"(a), "r"(parity) : "memory");
        if (done) return;
    }
    __trap();
}
__device__ __forceinline__ void tma_load_3d(void *dst_smem, const void *tmap, int c0, int c1, int c2, unsigned long long *bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(smem_u32(dst_smem)), "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}

// Programmatic dependent launch: let the next step's grid become resident while this one drains, and
// wait for the previous grid (and its memory) before touching anything it wrote.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

__device__ __forceinline__ float2 ldcs2(const float *p) { return __ldcs(reinterpret_cast<const float2 *>(p)); }
__device__ __forceinline__ void stcs2(float *p, float2 v) { __stcs(reinterpret_cast<float2 *>(p), v); }

__device__ __forceinline__ unsigned long long gtimer() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
// Timing experiments exist in -DRTM_DEBUG builds only (paper_2201_06914_b200/build.py: RTM_DEBUG=1 in the environment);
// the product library has neither the switches nor the stamps.
#ifdef RTM_DEBUG
#define DBG_STAMP(a, slot)                                                                  \
    do {                                                                                    \
        if (((a).dbg & 16) && threadIdx.x == 0 && threadIdx.y == 0 && blockIdx.x < 1024)    \
            (a).dbg_ts[blockIdx.x * 8 + (slot)] = gtimer();                                 \
    } while (0)
#define DBG_SKIP_STENCIL(a) (((a).dbg & 3) == 2)
#else
#define DBG_STAMP(a, slot) do { } while (0)
#define DBG_SKIP_STENCIL(a) false
#endif

// Flush role (time-blocked probing): PZ[k][x] += sum_{j<n} Z[n_j][k] hist[j][x] for this block's share of
// the slice, one float2 of x per thread; T history values stay in registers while r planes stream through.
template <int TM, int DEPTH = 1>
__device__ __forceinline__ void flush_role(const StepArgs &a, float *sz, int tid, int nthreads, int block) {
    const Layout &L = a.L;
    const int zr = a.zr, n = a.fl_n, r = a.r;
    for (int i = tid; i < TM * zr; i += nthreads) {
        const int j = i / zr, k = i - j * zr;
        sz[i] = j < n ? a.fl_Z0[j * a.fl_zstep + k] : 0.0f;
    }
    __syncthreads();
    // The history being flushed was written at least two launches ago whenever fl_nowait is set (the host schedules
    // the slices on slots >= 1 of the time block) and the stencil blocks release their dependents only after their
    // own wait, so every launch <= n-2 is complete when a block of launch n runs: no wait needed, and the role
    // overlaps with the previous step instead of starting behind it.
    DBG_STAMP(a, 0);
    if (!a.fl_nowait) pdl_wait();
    DBG_STAMP(a, 2);
    const int np = L.upz / 2;
    for (long long t = a.fl_q0 + (long long)block * nthreads + tid; t < a.fl_q1; t += (long long)a.fl_blocks * nthreads) {
        const long long row = t / np;
        const int iz = (int)(t - row * np) * 2;
        if (iz >= L.nz) continue;
        const long long o = row * L.upz + iz;
        float2 h[TM];
#pragma unroll
        for (int j = 0; j < TM; j++) h[j] = j < n ? ldcs2(a.fl_hist + j * a.pNu + o) : make_float2(0.f, 0.f);
        float *p = a.PZ + o;
        // software-pipelined over groups of 4 planes, DEPTH groups in flight: the loads of later groups are issued
        // BEFORE the stores of the current one (the compiler cannot hoist them itself: it cannot prove the planes do
        // not alias).  DEPTH 2 did not pay inside the 64-register budget of the 256-thread kernels (DEPTH 1 there);
        // the 128-thread 2D kernel uses 2 with T = 32.
        constexpr int G = 4;
        float2 ring[DEPTH][G];
#pragma unroll
        for (int s = 0; s < DEPTH; s++)
#pragma unroll
            for (int i = 0; i < G; i++)
                ring[s][i] = (s * G + i < r) ? ldcs2(p + (long long)(s * G + i) * a.pNu) : make_float2(0.f, 0.f);
        for (int kk = 0; kk < r; kk += G * DEPTH) {   // Z rows are zero-padded to zr (multiple of 8)
#pragma unroll
            for (int s = 0; s < DEPTH; s++) {
                const int k = kk + s * G;
                if (k >= r) break;
                float2 acc[G];
#pragma unroll
                for (int i = 0; i < G; i++) acc[i] = ring[s][i];
#pragma unroll
                for (int i = 0; i < G; i++) {
                    const int kn = k + G * DEPTH + i;
                    ring[s][i] = (kn < r) ? ldcs2(p + (long long)kn * a.pNu) : make_float2(0.f, 0.f);
                }
                // one FFMA2 per (plane, history slot): both x lanes of the float2 in one issue slot, each lane rounded
                // exactly like the scalar FMA it replaces
                f32x2 ap[G];
#pragma unroll
                for (int i = 0; i < G; i++) ap[i] = pk(acc[i].x, acc[i].y);
#pragma unroll
                for (int j = 0; j < TM; j++) {
                    const float4 z = ld4(sz + j * zr + k);
                    const f32x2 hp = pk(h[j].x, h[j].y);
                    ap[0] = fma2(pk(z.x, z.x), hp, ap[0]);
                    ap[1] = fma2(pk(z.y, z.y), hp, ap[1]);
                    ap[2] = fma2(pk(z.z, z.z), hp, ap[2]);
                    ap[3] = fma2(pk(z.w, z.w), hp, ap[3]);
                }
#pragma unroll
                for (int i = 0; i < G; i++) {
                    upk(ap[i], acc[i].x, acc[i].y);
                    if (k + i < r) stcs2(p + (long long)(k + i) * a.pNu, acc[i]);
                }
            }
        }
    }
    DBG_STAMP(a, 6);
}

// Same role with one float4 of x per thread (fewer, fatter threads: used by the 2D streaming kernel, whose
// stencil threads need ~120 registers anyway).  The Z rows are staged BEFORE griddepcontrol.wait (static
// data); the history of the previous time block is only touched after it.  Pipelined over groups of 2 planes.
template <int TM>
__device__ __forceinline__ void flush_role4(const StepArgs &a, float *sz, int tid, int nthreads, int block) {
    const Layout &L = a.L;
    const int zr = a.zr, n = a.fl_n, r = a.r;
    for (int i = tid; i < TM * zr; i += nthreads) {
        const int j = i / zr, k = i - j * zr;
        sz[i] = j < n ? a.fl_Z0[j * a.fl_zstep + k] : 0.0f;
    }
    __syncthreads();
    DBG_STAMP(a, 0);
    if (!a.fl_nowait) pdl_wait();   // see flush_role
    DBG_STAMP(a, 2);
    const int nq = L.upz / 4;
    for (long long t = a.fl_q0 + (long long)block * nthreads + tid; t < a.fl_q1; t += (long long)a.fl_blocks * nthreads) {
        const long long row = t / nq;
        const int iz = (int)(t - row * nq) * 4;
        if (iz >= L.nz) continue;
        const long long o = row * L.upz + iz;
        float4 h[TM];
#pragma unroll
        for (int j = 0; j < TM; j++) h[j] = j < n ? ldcs4(a.fl_hist + j * a.pNu + o) : make_float4(0.f, 0.f, 0.f, 0.f);
        float *p = a.PZ + o;
        // The plane loop is a chain of DRAM round trips (load - FMA - store per group): with one group of look-ahead
        // the role needed 1 + r/2 round trips per thread (measured 15 us at c1, longer than the stencil blocks it
        // shares the launch with).  Three groups of two planes are kept in flight instead.
        constexpr int G = 2, DEPTH = 3;
        float4 ring[DEPTH][G];
#pragma unroll
        for (int s = 0; s < DEPTH; s++)
#pragma unroll
            for (int i = 0; i < G; i++)
                ring[s][i] = (s * G + i < r) ? ldcs4(p + (long long)(s * G + i) * a.pNu) : make_float4(0.f, 0.f, 0.f, 0.f);
        for (int kk = 0; kk < r; kk += G * DEPTH) {   // Z rows are zero-padded to zr (multiple of 8)
#pragma unroll
            for (int s = 0; s < DEPTH; s++) {
                const int k = kk + s * G;
                if (k >= r) break;
                float4 acc[G];
#pragma unroll
                for (int i = 0; i < G; i++) acc[i] = ring[s][i];
#pragma unroll
                for (int i = 0; i < G; i++) {
                    const int kn = k + G * DEPTH + i;
                    ring[s][i] = (kn < r) ? ldcs4(p + (long long)kn * a.pNu) : make_float4(0.f, 0.f, 0.f, 0.f);
                }
                f32x2 alo[G], ahi[G];   // packed FMAs, see flush_role
#pragma unroll
                for (int i = 0; i < G; i++) { alo[i] = pk(acc[i].x, acc[i].y); ahi[i] = pk(acc[i].z, acc[i].w); }
#pragma unroll
                for (int j = 0; j < TM; j++) {
                    const float2 z = *reinterpret_cast<const float2 *>(sz + j * zr + k);
                    const f32x2 hlo = pk(h[j].x, h[j].y), hhi = pk(h[j].z, h[j].w);
                    const f32x2 z0 = pk(z.x, z.x), z1 = pk(z.y, z.y);
                    alo[0] = fma2(z0, hlo, alo[0]); ahi[0] = fma2(z0, hhi, ahi[0]);
                    alo[1] = fma2(z1, hlo, alo[1]); ahi[1] = fma2(z1, hhi, ahi[1]);
                }
#pragma unroll
                for (int i = 0; i < G; i++) {
                    upk(alo[i], acc[i].x, acc[i].y); upk(ahi[i], acc[i].z, acc[i].w);
                    if (k + i < r) stcs4(p + (long long)(k + i) * a.pNu, acc[i]);
                }
            }
        }
    }
    DBG_STAMP(a, 6);
}

__device__ __forceinline__ float k1_of(float s) { return s == 0.0f ? 1.0f : (1.0f - s) / (1.0f + s); }
// Deferred receiver sampling: the first ceil(nsmp/nthreads) blocks (linear order) take one point
// per thread (a4: d[j] = scale * sum_c w_c u[corner]; TTI samples p + r).
__device__ __forceinline__ void sample_points(const StepArgs &a, int lin_block, int nthreads, int tid) {
    if (a.smp_out == nullptr) return;
    long long j = (long long)lin_block * nthreads + tid;
    if (j >= a.nsmp) return;
    float acc = 0.0f;
    for (int c = 0; c < a.nc; c++) {
        float w = a.smp_w[j * a.nc + c];
        if (w != 0.0f) {
            int i = a.smp_idx[j * a.nc + c];
            float v = a.u0[i];
            if (a.u1) v += a.u1[i];
            acc = fmaf(w, v, acc);
        }
    }
    a.smp_out[j] = a.smp_scale * acc;
}

// Fused injection for one z-quad at row `row` (a3): adds K2 * scale * w * val to the increments.
__device__ __forceinline__ void inject_quad(const StepArgs &a, long long row, int jz, const float k2[4], float add[4]) {
    int e0 = a.row_start[row], e1 = a.row_start[row + 1];
    for (int e = e0; e < e1; e++) {
        InjEntry en = a.ent[e];
        int dz = en.jz - jz;
        if (dz >= 0 && dz < 4) {
            float v = a.inj_scale * en.w * a.inj_val[en.id];
#pragma unroll
            for (int q = 0; q < 4; q++)
                if (q == dz) add[q] = fmaf(k2[q], v, add[q]);
        }
    }
}

// Fused probe for one z-quad (a5): PZ[k][x] += Z[k] * v for k < r.  p points at plane 0.  Zrow is padded
// with zeros to a multiple of 8.  The update is a chain of DRAM round trips per thread (load - 4 FMA - store per
// plane), so its bandwidth is its bytes in flight: PQ_DEPTH groups of 4 planes are kept in flight (the loads of
// later groups are issued before the stores of the current one; see flush_role).
// Measured (per-step fused schedule): 2D acoustic 68.5 us at DEPTH 1 / 4 blocks per SM against 72.9 us at DEPTH 2 /
// 3 blocks; TTI 246 us against 218 us: the kernels pick their own depth.
// Per-step fused probing: ask L2 for this thread's 16 bytes of every probe plane at the START of the step kernel, so that
// the DRAM reads of the planes are spread over the stencil phase instead of starting behind it (the planes are written
// by the previous launch; L2 is the coherence point, so the request may even precede griddepcontrol.wait).
__device__ __forceinline__ void prefetch_planes(const float *p, long long Nu, int r) {
    for (int k = 0; k < r; k++) asm volatile("prefetch.global.L2 [%0];" ::"l"(p + (long long)k * Nu));
}

template <int DEPTH>
__device__ __forceinline__ void probe_quad(float *p, long long Nu, const float *__restrict__ Zrow, int r, float4 v) {
    constexpr int G = 4;
    float4 ring[DEPTH][G];
#pragma unroll
    for (int s = 0; s < DEPTH; s++)
#pragma unroll
        for (int i = 0; i < G; i++)
            ring[s][i] = (s * G + i < r) ? ldcs4(p + (long long)(s * G + i) * Nu) : make_float4(0.f, 0.f, 0.f, 0.f);
    for (int kk = 0; kk < r; kk += G * DEPTH) {
#pragma unroll
        for (int s = 0; s < DEPTH; s++) {
            const int k = kk + s * G;
            if (k >= r) break;
            float4 acc[G];
#pragma unroll
            for (int i = 0; i < G; i++) acc[i] = ring[s][i];
#pragma unroll
            for (int i = 0; i < G; i++) {
                const int kn = k + G * DEPTH + i;
                ring[s][i] = (kn < r) ? ldcs4(p + (long long)kn * Nu) : make_float4(0.f, 0.f, 0.f, 0.f);
            }
            const float4 z4 = ldg4(Zrow + k);
            const float z[4] = {z4.x, z4.y, z4.z, z4.w};
#pragma unroll
            for (int i = 0; i < G; i++) {
                acc[i].x = fmaf(z[i], v.x, acc[i].x);
                acc[i].y = fmaf(z[i], v.y, acc[i].y);
                acc[i].z = fmaf(z[i], v.z, acc[i].z);
                acc[i].w = fmaf(z[i], v.w, acc[i].w);
            }
#pragma unroll
            for (int i = 0; i < G; i++)
                if (k + i < r) stcs4(p + (long long)(k + i) * Nu, acc[i]);
        }
    }
}

}  // namespace rtm
