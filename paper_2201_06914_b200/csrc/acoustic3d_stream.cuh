// acoustic3d_stream.cuh -- 3D isotropic acoustic time step (a1) for time-blocked probing: 2.5D blocking.
//
// Block = 256 threads = a (y, z) tile of 8 x 128 points, one z-quad (float4) per thread, streaming along the
// slow axis x over a chunk of S3_XCH planes.
//   - x neighbours: a 9-deep register queue per thread that slides one plane per iteration (1 new LDG.128 per
//     plane instead of 8);
//   - y and z neighbours: the current plane of the tile (+ halo of 4 in y and z) staged in shared memory,
//     double-buffered, one __syncthreads per plane;
//   - the operands of plane p+1 (queue head, halo quads, K2, du, damping) are requested before the arithmetic
//     of plane p.
// Per plane and quad: 5 LDG.128 + 2 STS.128 + 10 LDS.128 + 3 STG.128 + ~210 flops, against 23 LDG.128 of the
// plain kernel; DRAM traffic stays at the algorithmic 20 B/point (u, du read; u', du' written; K2) because the
// x re-reads of neighbouring chunks and the y/z halos hit L2.
//
// Fused as in the 2D kernel: damping through per-axis K1 tables, source injection (a3; the block's injection
// amounts are looked up by all 256 threads in parallel before griddepcontrol.wait), deferred receiver sampling
// (a4), history store for the probe (a5), and the flush role in the leading blocks of the launch.
#pragma once
#include "common.cuh"

namespace rtm {

constexpr int S3_TY = 8, S3_TZ = 128;
constexpr int S3_PITCH = S3_TZ + 8;     // floats per smem row: [z halo 4 | 128 | z halo 4]
constexpr int S3_ROWS = S3_TY + 8;      // y halo 4 on both sides
constexpr int S3_XCH = 32;              // planes per chunk
constexpr int S3_INJCAP = 512;          // injection amounts (float4) a block can stage
constexpr int S3_SMEM = (2 * S3_ROWS * S3_PITCH) * 4 + S3_INJCAP * 16;

// sum of the injection entries of padded row `row` that fall into the z-quad starting at jz (a3)
__device__ __forceinline__ float4 inject_lookup(const StepArgs &a, long long row, int jz) {
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    const int e0 = a.row_start[row], e1 = a.row_start[row + 1];
    for (int e = e0; e < e1; e++) {
        const InjEntry en = a.ent[e];
        const int dz = en.jz - jz;
        if (dz >= 0 && dz < 4) {
            const float v = a.inj_scale * en.w * a.inj_val[en.id];
#pragma unroll
            for (int q = 0; q < 4; q++)
                if (q == dz) acc[q] += v;
        }
    }
    return make_float4(acc[0], acc[1], acc[2], acc[3]);
}

template <int TM>
__global__ void __launch_bounds__(256, 2) acoustic3d_stream_kernel(const __grid_constant__ StepArgs a) {
    extern __shared__ __align__(16) float dyn_smem[];
    const Layout &L = a.L;
    const int tid = threadIdx.x;
    pdl_launch_dependents();
    if (blockIdx.x < (unsigned)a.fl_blocks) {
        flush_role<TM>(a, dyn_smem, tid, 256, blockIdx.x);
        return;
    }
    const unsigned lin_block = blockIdx.x - a.fl_blocks;
    const int tx = tid & 31, ty = tid >> 5;
    const unsigned bz = lin_block % a.gx, t1 = lin_block / a.gx;
    const unsigned by = t1 % a.gy, ch = t1 / a.gy;
    const int jz = (int)bz * S3_TZ + tx * 4, jy = (int)by * S3_TY + ty;
    const int x0 = (int)ch * S3_XCH;
    const int nplanes = min(S3_XCH, L.Px - x0);
    const bool act = jz < L.Pz && jy < L.Py;

    float *plane = dyn_smem;                                                   // [2][S3_ROWS][S3_PITCH]
    float4 *injs = reinterpret_cast<float4 *>(dyn_smem + 2 * S3_ROWS * S3_PITCH);   // [S3_INJCAP]

    // ---- prologue on static data (before the grid dependency is resolved) ----------------------------------
    // injection: all (plane, row, z-quad) triples of this block's tile that intersect the bounding box of the
    // geometry, one lookup per thread, results in shared memory (inj_mode 1); a geometry too dense for the
    // staging buffer is looked up in the plane loop instead (inj_mode 2)
    const int zq0 = max((int)bz * (S3_TZ / 4), a.bz0 >> 2), zq1 = min((int)bz * (S3_TZ / 4) + S3_TZ / 4 - 1, a.bz1 >> 2);
    const int r0 = max((int)by * S3_TY, a.by0), r1 = min(min((int)by * S3_TY + S3_TY - 1, a.by1), L.Py - 1);
    const int p0 = max(x0, a.bx0), p1 = min(x0 + nplanes - 1, a.bx1);
    const int nzq = zq1 - zq0 + 1, nr = r1 - r0 + 1, npl = p1 - p0 + 1;
    const int total = (nzq > 0 && nr > 0 && npl > 0) ? nzq * nr * npl : 0;
    const int inj_mode = total == 0 ? 0 : (total <= S3_INJCAP ? 1 : 2);
    if (inj_mode == 1) {
        for (int idx = tid; idx < total; idx += 256) {
            const int zq = zq0 + idx % nzq, rr = r0 + (idx / nzq) % nr, pp = p0 + idx / (nzq * nr);
            injs[idx] = inject_lookup(a, (long long)pp * L.Py + rr, zq * 4);
        }
    }
    const bool my_hit = inj_mode != 0 && act && (jz >> 2) >= zq0 && (jz >> 2) <= zq1 && jy >= r0 && jy <= r1;
    const int my_inj = ((jz >> 2) - zq0) + (jy - r0) * nzq;   // + (plane - p0) * nzq * nr

    // per-thread damping tables of the y and z axes
    float dzv[4] = {0.f, 0.f, 0.f, 0.f}, k1z[4] = {1.f, 1.f, 1.f, 1.f};
    float syv = 0.f, k1yv = 1.f;
    if (act) {
        const float4 d4 = ld4(a.dampz + jz), k4 = ld4(a.k1z + jz);
        dzv[0] = d4.x; dzv[1] = d4.y; dzv[2] = d4.z; dzv[3] = d4.w;
        k1z[0] = k4.x; k1z[1] = k4.y; k1z[2] = k4.z; k1z[3] = k4.w;
        syv = a.dampy[jy];
        k1yv = a.k1y[jy];
    }
    const bool zdamp = (dzv[0] != 0.f) | (dzv[1] != 0.f) | (dzv[2] != 0.f) | (dzv[3] != 0.f);

    pdl_wait();   // from here on the previous step's fields are complete and visible
    sample_points(a, lin_block, 256, tid);

    const float *__restrict__ u0 = a.u0;
    const float *__restrict__ K2 = a.K2;
    float *__restrict__ n0 = a.n0;
    float *d0 = a.d0;

    // what this thread may load: its centre quad (also when it only feeds a neighbour's halo) ...
    const bool ld_c = jz + 8 <= L.pz && jy < L.Py + 4;
    // ... one quad of the y halo (rows -4..-1 and 8..11 of the tile) ...
    const int hrow = ty < 4 ? ty : ty + S3_TY;                 // smem row of the halo quad
    const int jyh = (int)by * S3_TY + hrow - 4;
    const bool ld_h = jz + 8 <= L.pz && jyh < L.Py + 4;
    // ... and, for the first / last lane of a row, one quad of the z halo
    const bool zl = tx == 0, zr_ = tx == 31;
    const bool ld_z = (zl || (zr_ && jz + 12 <= L.pz)) && jy < L.Py + 4;

    const long long sx = L.sx;
    const long long oc = L.org + (long long)x0 * sx + (long long)jy * L.sy + jz;
    const float *pc = u0 + oc;                                  // centre quad, plane x0
    const float *phh = u0 + L.org + (long long)x0 * sx + (long long)jyh * L.sy + jz;
    const float *pk = K2 + oc;
    float *pd = d0 + oc;
    float *pn = n0 + oc;
    const int iz = jz - L.nb, iy = jy - L.nby;
    const bool phys_yz = act && iz >= 0 && iz < L.nz && iy >= 0 && iy < L.ny && a.hist != nullptr;
    float *ph = a.hist + (((long long)(x0 - L.nb) * L.ny + iy) * L.upz + iz);   // dereferenced inside the physical grid only
    const long long hstep = (long long)L.ny * L.upz;

    const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
    float4 q[9];
#pragma unroll
    for (int i = 0; i < 9; i++) q[i] = ld_c ? ld4(pc + (i - 4) * sx) : zero4;
    float4 hy = ld_h ? ld4(phh) : zero4;
    float4 hz = ld_z ? ld4(pc + (zl ? -4 : 4)) : zero4;
    float4 k24 = act ? ld4(pk) : zero4, du4 = act ? ld4(pd) : zero4;
    float sxd = a.dampx[x0], k1x = a.k1x[x0];

    float *srow = plane + (ty + 4) * S3_PITCH + 4 + tx * 4;    // this thread's centre slot in buffer 0
    float *shal = plane + hrow * S3_PITCH + 4 + tx * 4;        // its y-halo slot
    constexpr int BUF = S3_ROWS * S3_PITCH;

#pragma unroll 1
    for (int p = 0; p < nplanes; p++) {
        const int b = (p & 1) * BUF;
        const float4 c = q[4];
        st4(srow + b, c);
        st4(shal + b, hy);
        if (zl) st4(srow + b - 4, hz);
        if (zr_) st4(srow + b + 4, hz);
        __syncthreads();

        const float k2[4] = {k24.x, k24.y, k24.z, k24.w};
        const float du[4] = {du4.x, du4.y, du4.z, du4.w};
        const float sxc = sxd, k1xc = k1x;
        float4 qn = zero4;
        if (p + 1 < nplanes) {   // operands of plane p+1, requested before the arithmetic of plane p
            qn = ld_c ? ld4(pc + 5 * sx) : zero4;
            hy = ld_h ? ld4(phh + sx) : zero4;
            hz = ld_z ? ld4(pc + sx + (zl ? -4 : 4)) : zero4;
            if (act) { k24 = ld4(pk + sx); du4 = ld4(pd + sx); }
            sxd = a.dampx[x0 + p + 1];
            k1x = a.k1x[x0 + p + 1];
        }

        const float4 zm = ld4(srow + b - 4), zp = ld4(srow + b + 4);
        const float win[12] = {zm.x, zm.y, zm.z, zm.w, c.x, c.y, c.z, c.w, zp.x, zp.y, zp.z, zp.w};
        const float cc[4] = {c.x, c.y, c.z, c.w};
        float lap[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int j = 4; j >= 1; j--) {   // small weights first
            const float4 XP = q[4 + j], XM = q[4 - j];
            const float4 YP = ld4(srow + b + j * S3_PITCH), YM = ld4(srow + b - j * S3_PITCH);
            const float xs[4] = {(XP.x - c.x) + (XM.x - c.x), (XP.y - c.y) + (XM.y - c.y),
                                 (XP.z - c.z) + (XM.z - c.z), (XP.w - c.w) + (XM.w - c.w)};
            const float ys[4] = {(YP.x - c.x) + (YM.x - c.x), (YP.y - c.y) + (YM.y - c.y),
                                 (YP.z - c.z) + (YM.z - c.z), (YP.w - c.w) + (YM.w - c.w)};
            const float w = w2(j);
#pragma unroll
            for (int e = 0; e < 4; e++) {
                const float s = (((win[4 + e + j] - cc[e]) + (win[4 + e - j] - cc[e])) + xs[e]) + ys[e];
                lap[e] = fmaf(w, s, lap[e]);
            }
        }
        float d[4];
        const float sxy = sxc + syv;
        if (sxy == 0.f && !zdamp) {
#pragma unroll
            for (int e = 0; e < 4; e++) d[e] = fmaf(k2[e], lap[e], du[e]);          // K1 = 1 exactly
        } else {
            // one damping axis: its table; several: (1 - s) / (1 + s) with s = (sx + sy) + sz
            const float k1xy = sxc == 0.f ? k1yv : (syv == 0.f ? k1xc : k1_of(sxy));
#pragma unroll
            for (int e = 0; e < 4; e++) {
                const float k1 = sxy == 0.f ? k1z[e] : (dzv[e] == 0.f ? k1xy : k1_of(sxy + dzv[e]));
                d[e] = fmaf(k1, du[e], k2[e] * lap[e]);
            }
        }
        const int jx = x0 + p;
        if (my_hit && jx >= p0 && jx <= p1) {   // a3: K2 * scale * w * val
            const float4 iv = inj_mode == 1 ? injs[my_inj + (jx - p0) * nzq * nr]
                                            : inject_lookup(a, (long long)jx * L.Py + jy, jz);
            d[0] = fmaf(k2[0], iv.x, d[0]);
            d[1] = fmaf(k2[1], iv.y, d[1]);
            d[2] = fmaf(k2[2], iv.z, d[2]);
            d[3] = fmaf(k2[3], iv.w, d[3]);
        }
        if (act) {
            float4 dn = make_float4(d[0], d[1], d[2], d[3]);
            float4 un = make_float4(cc[0] + d[0], cc[1] + d[1], cc[2] + d[2], cc[3] + d[3]);
            if (jz + 3 >= L.Pz) {   // ragged quad at the end of a row: keep the halo zero
                if (jz + 1 >= L.Pz) { dn.y = 0.f; un.y = 0.f; }
                if (jz + 2 >= L.Pz) { dn.z = 0.f; un.z = 0.f; }
                dn.w = 0.f; un.w = 0.f;
            }
            st4(pd, dn);
            st4(pn, un);
            if (phys_yz && (unsigned)(jx - L.nb) < (unsigned)L.nx) stcs4(ph, un);
        }
        // slide the x queue by one plane
#pragma unroll
        for (int i = 0; i < 8; i++) q[i] = q[i + 1];
        q[8] = qn;
        pc += sx; phh += sx; pk += sx; pd += sx; pn += sx; ph += hstep;
    }
}

}  // namespace rtm
