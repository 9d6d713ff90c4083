// acoustic3d_stream.cuh -- 3D isotropic acoustic time step (a1) for time-blocked probing: 2.5D blocking fed by the
// tensor memory accelerator.
//
// Block = 256 threads = a (y, z) tile of 8 x 128 points, one z-quad (float4) per thread, streaming along the
// slow axis x over a chunk of S3_XCH planes.
//   - every tile comes through TMA (cp.async.bulk.tensor, SASS UTMALDG): ONE thread asks for the haloed 16 x 136 box
//     of u of plane p+4+D and the 8 x 128 boxes of K2 and du of plane p+D while plane p is computed; the bytes land
//     in rings in shared memory and are counted on an mbarrier per group.  No thread spends instructions on
//     addresses, bounds or zero fill (the round-1 cp.async version spent ~70 of its ~450 instructions per plane and
//     quad on exactly that, plus the registers that forced the compiler to recompute loop invariants); boxes that
//     stick out of the allocation are zero-filled by the copy engine, which is the boundary condition (C8);
//   - x neighbours: a 9-deep register queue per thread that slides one plane per iteration and is fed from the
//     ring when a plane arrives;
//   - y and z neighbours: read from the ring slot of the current plane (halo of 4 in y and z);
//   - one __syncthreads per plane: it frees the slots the next request overwrites.
// Per plane and quad: 13 LDS.128 + 3 STG.128, arithmetic in packed fp32x2 (FADD2 / FFMA2).  DRAM traffic stays at the
// algorithmic 20 B/point (u, du read; u', du' written; K2): the x re-reads of neighbouring chunks and the y/z halos
// hit L2.
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
constexpr int S3_D = 3;                 // prefetch distance in planes
constexpr int S3_NU = 8;                // u ring slots  = 5 + S3_D (planes p .. p+4+D)
constexpr int S3_NK = 4;                // K2 / du ring slots = S3_D + 1
constexpr int S3_TILE = S3_ROWS * S3_PITCH;      // floats per haloed u tile
constexpr int S3_CT = S3_TY * S3_TZ;             // floats per K2 / du tile
constexpr int S3_INJCAP = 512;          // injection amounts (float4) a block can stage
constexpr int S3_NB = 4;                // mbarriers: groups p .. p+D are in flight
constexpr int S3_SMEM = (S3_NU * S3_TILE + 2 * S3_NK * S3_CT) * 4 + S3_INJCAP * 16 + S3_NB * 8;
static_assert(S3_NU == 5 + S3_D && S3_NK == S3_D + 1 && S3_NB == S3_D + 1, "ring sizes follow the prefetch distance");
static_assert((S3_TILE * 4) % 128 == 0 && (S3_CT * 4) % 128 == 0, "TMA destinations stay 128-byte aligned");

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

template <int TM, bool PK>
__global__ void __launch_bounds__(256, 2) acoustic3d_stream_kernel(const __grid_constant__ StepArgs a) {
    extern __shared__ __align__(128) float dyn_smem[];
    const Layout &L = a.L;
    const int tid = threadIdx.x;
    if (blockIdx.x < (unsigned)a.fl_blocks) {
        pdl_launch_dependents();
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

    float4 *injs = reinterpret_cast<float4 *>(dyn_smem + S3_NU * S3_TILE + 2 * S3_NK * S3_CT);   // [S3_INJCAP], behind the rings
    unsigned long long *bars = reinterpret_cast<unsigned long long *>(injs + S3_INJCAP);          // [S3_NB] mbarriers
    if (tid == 0) {
        for (int i = 0; i < S3_NB; i++) mbar_init(bars + i, 1);   // one arrival (thread 0's expect_tx) + the bytes
        mbar_fence_init();
    }

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

    __syncthreads();   // the mbarriers are initialised (and the staged injection amounts visible) before anybody waits
    pdl_wait();   // from here on the previous step's fields are complete and visible
    pdl_launch_dependents();   // only now: lets the next step's flush role run without a wait (see flush_role)
    sample_points(a, lin_block, 256, tid);

    const float *__restrict__ u0 = a.u0;
    const float *__restrict__ K2 = a.K2;
    float *__restrict__ n0 = a.n0;
    float *d0 = a.d0;

    const long long sx = L.sx;
    const long long oc = L.org + (long long)x0 * sx + (long long)jy * L.sy + jz;
    const float *pc = u0 + oc;                                  // centre quad, plane x0
    const int iz = jz - L.nbz, iy = jy - L.nby;
    const bool phys_yz = act && iz >= 0 && iz < L.nz && iy >= 0 && iy < L.ny && a.hist != nullptr;
    const long long hstep = (long long)L.ny * L.upz;

    float *Ub = dyn_smem;                                        // [S3_NU][S3_ROWS][S3_PITCH]
    float *Kb = Ub + S3_NU * S3_TILE;                            // [S3_NK][S3_TY][S3_TZ]
    float *Db = Kb + S3_NK * S3_CT;
    const int o_c = (ty + 4) * S3_PITCH + 4 + tx * 4;            // this thread's centre slot inside a u tile
    const int o_k = tid * 4;
    const bool ld_c = jz + 8 <= L.pz && jy < L.Py + 4;           // its centre quad exists in the allocation

    // Group g = the haloed u tile of plane g+4 (group 0: planes 0..4) and the K2 / du tiles of plane g, relative to
    // x0; planes 0 .. nplanes+3 of u are needed, so a group is needed iff g < nplanes.  Tensor coordinates are
    // (z, y, x) counted from the first allocated float of a field: padded index + halo (4 on every axis here).
    const char *tmaps = (const char *)a.tmaps;
    const void *tm_u = tmaps + 128 * a.tm_u, *tm_k = tmaps + 256, *tm_d = tmaps + 384;
    const int cz = (int)bz * S3_TZ, cy = (int)by * S3_TY, cx = x0 + 4;      // the box of u starts 4 before the tile
    auto issue = [&](int g) {                                    // thread 0 only
        if (g >= nplanes) return;
        unsigned long long *bar = bars + (g & (S3_NB - 1));
        mbar_arrive_expect_tx(bar, (unsigned)((g == 0 ? 5 : 1) * S3_TILE * 4 + 2 * S3_CT * 4));
        if (g == 0)
            for (int pl = 0; pl < 4; pl++) tma_load_3d(Ub + pl * S3_TILE, tm_u, cz, cy, cx + pl, bar);
        tma_load_3d(Ub + ((g + 4) & (S3_NU - 1)) * S3_TILE, tm_u, cz, cy, cx + g + 4, bar);
        tma_load_3d(Kb + (g & (S3_NK - 1)) * S3_CT, tm_k, cz + 4, cy + 4, cx + g, bar);
        tma_load_3d(Db + (g & (S3_NK - 1)) * S3_CT, tm_d, cz + 4, cy + 4, cx + g, bar);
    };
    if (tid == 0)
        for (int g = 0; g < S3_D; g++) issue(g);

    // running output pointers (this thread's quad of plane x0 + p)
    float *pd = d0 + oc;
    float *pn = n0 + oc;
    float *ph = a.hist + (((long long)(x0 - L.nb) * L.ny + iy) * L.upz + iz);   // dereferenced inside the physical grid only

    const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
    // (Unrolling the plane loop by 8 with a circular queue of 8 register quads removes the 32 moves per plane that slide
    // this queue and makes every ring offset a constant, but the body grows 8-fold (142 KB of SASS) and the launch gets
    // slower: c4 0.749 ms per step against 0.677.  Kept rolled.)
    float4 q[9];   // planes p-4 .. p+4 of this thread's quad; q[8] is filled from the ring at the top of iteration p
#pragma unroll
    for (int i = 0; i < 8; i++) q[i] = ld_c ? ld4(pc + (i - 4) * sx) : zero4;

    typedef V2<PK> V;
    typedef typename V::T P2;
    float sxn = a.dampx[x0], k1xn = a.k1x[x0];   // x damping of the next plane, fetched one iteration ahead
#pragma unroll 1
    for (int p = 0; p < nplanes; p++) {
        __syncthreads();             // nobody reads the slots (and the mbarrier) the next group overwrites any more
        if (tid == 0) issue(p + S3_D);
        mbar_wait(bars + (p & (S3_NB - 1)), (unsigned)(p / S3_NB) & 1u);   // group p has landed: u plane p+4, K2 / du plane p

        const float *U0 = Ub + (p & (S3_NU - 1)) * S3_TILE + o_c;            // current plane, centre slot
        q[8] = ld4(Ub + ((p + 4) & (S3_NU - 1)) * S3_TILE + o_c);
        const float4 c = q[4];
        const float4 k24c = act ? ld4(Kb + (p & (S3_NK - 1)) * S3_CT + o_k) : zero4;
        const float4 du4c = act ? ld4(Db + (p & (S3_NK - 1)) * S3_CT + o_k) : zero4;
        const int jx = x0 + p;
        const float sxc = sxn, k1xc = k1xn;
        sxn = a.dampx[jx + 1];   // tables are padded: jx + 1 <= Px is readable
        k1xn = a.k1x[jx + 1];

        const float4 zm = ld4(U0 - 4), zp = ld4(U0 + 4);
        const float win[12] = {zm.x, zm.y, zm.z, zm.w, c.x, c.y, c.z, c.w, zp.x, zp.y, zp.z, zp.w};
        const float cc[4] = {c.x, c.y, c.z, c.w};
        // Laplacian in the difference form, two z points per instruction (FADD2 / FFMA2); same operations in
        // the same order per point as the scalar kernels: s = ((z part + x part) + y part), lap = fma(w, s, lap)
        const P2 clo = V::mk(c.x, c.y), chi = V::mk(c.z, c.w);
        P2 llo = V::mk(0.f, 0.f), lhi = llo;
#pragma unroll
        for (int j = 4; j >= 1; j--) {   // small weights first
            const float4 XP = q[4 + j], XM = q[4 - j];
            const float4 YP = ld4(U0 + j * S3_PITCH), YM = ld4(U0 - j * S3_PITCH);
            const P2 xlo = V::dd(V::mk(XP.x, XP.y), V::mk(XM.x, XM.y), clo), xhi = V::dd(V::mk(XP.z, XP.w), V::mk(XM.z, XM.w), chi);
            const P2 ylo = V::dd(V::mk(YP.x, YP.y), V::mk(YM.x, YM.y), clo), yhi = V::dd(V::mk(YP.z, YP.w), V::mk(YM.z, YM.w), chi);
            P2 zlo, zhi;
            if (j % 2 == 0) {   // shifted z windows are register-pair aligned for even shifts only
                zlo = V::dd(V::mk(win[4 + j], win[5 + j]), V::mk(win[4 - j], win[5 - j]), clo);
                zhi = V::dd(V::mk(win[6 + j], win[7 + j]), V::mk(win[6 - j], win[7 - j]), chi);
            } else {
                float zs[4];
#pragma unroll
                for (int e = 0; e < 4; e++) zs[e] = (win[4 + e + j] - cc[e]) + (win[4 + e - j] - cc[e]);
                zlo = V::mk(zs[0], zs[1]);
                zhi = V::mk(zs[2], zs[3]);
            }
            const float w = w2(j);
            const P2 ww = V::mk(w, w);
            llo = V::fma(ww, V::add(V::add(zlo, xlo), ylo), llo);
            lhi = V::fma(ww, V::add(V::add(zhi, xhi), yhi), lhi);
        }
        const P2 k2lo = V::mk(k24c.x, k24c.y), k2hi = V::mk(k24c.z, k24c.w);
        const P2 dulo = V::mk(du4c.x, du4c.y), duhi = V::mk(du4c.z, du4c.w);
        P2 dlo, dhi;
        const float sxy = sxc + syv;
        if (sxy == 0.f && !zdamp) {
            dlo = V::fma(k2lo, llo, dulo);          // K1 = 1 exactly
            dhi = V::fma(k2hi, lhi, duhi);
        } else {
            // one damping axis: its table; several: (1 - s) / (1 + s) with s = (sx + sy) + sz
            const float k1xy = sxc == 0.f ? k1yv : (syv == 0.f ? k1xc : k1_of(sxy));
            float k1[4];
#pragma unroll
            for (int e = 0; e < 4; e++) k1[e] = sxy == 0.f ? k1z[e] : (dzv[e] == 0.f ? k1xy : k1_of(sxy + dzv[e]));
            dlo = V::fma(V::mk(k1[0], k1[1]), dulo, V::mul(k2lo, llo));
            dhi = V::fma(V::mk(k1[2], k1[3]), duhi, V::mul(k2hi, lhi));
        }
        if (my_hit && jx >= p0 && jx <= p1) {   // a3: K2 * scale * w * val
            const float4 iv = inj_mode == 1 ? injs[my_inj + (jx - p0) * nzq * nr]
                                            : inject_lookup(a, (long long)jx * L.Py + jy, jz);
            dlo = V::fma(k2lo, V::mk(iv.x, iv.y), dlo);
            dhi = V::fma(k2hi, V::mk(iv.z, iv.w), dhi);
        }
        if (act) {
            const P2 ulo = V::add(clo, dlo), uhi = V::add(chi, dhi);
            float4 dn, un;
            V::get(dlo, dn.x, dn.y); V::get(dhi, dn.z, dn.w);
            V::get(ulo, un.x, un.y); V::get(uhi, un.z, un.w);
            if (jz + 3 >= L.Pz) {   // ragged quad at the end of a row: keep the halo zero
                if (jz + 1 >= L.Pz) { dn.y = 0.f; un.y = 0.f; }
                if (jz + 2 >= L.Pz) { dn.z = 0.f; un.z = 0.f; }
                dn.w = 0.f; un.w = 0.f;
            }
            st4(pd, dn);
            st4(pn, un);
            if (phys_yz && (unsigned)(jx - L.nb) < (unsigned)L.nx) stcs4(ph, un);
        }
        pd += sx; pn += sx; ph += hstep;
        // slide the x queue by one plane
#pragma unroll
        for (int i = 0; i < 8; i++) q[i] = q[i + 1];
    }
}

}  // namespace rtm
