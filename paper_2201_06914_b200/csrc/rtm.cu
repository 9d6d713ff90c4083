// rtm.cu -- host side of the C ABI declared in include/rtm.h: context, workspace carving, geometry
// tables, time loops, image / gather launches.  All device arithmetic lives in the *.cuh kernels.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include <cuda.h>   // CUtensorMap (types only: the encoder is fetched through cudaGetDriverEntryPoint, no -lcuda)

#include "../../include/rtm.h"
#include "acoustic.cuh"
#include "acoustic2d_resident.cuh"
#include "acoustic2d_stream.cuh"
#include "acoustic3d_stream.cuh"
#include "image.cuh"
#include "tti.cuh"
#include "tti3d.cuh"

using namespace rtm;

static thread_local char g_cuda_err[256] = "";

#define CU(call)                                                                                   \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess) {                                                                   \
            snprintf(g_cuda_err, sizeof g_cuda_err, "%s: %s (%s:%d)", #call, cudaGetErrorString(e_), \
                     __FILE__, __LINE__);                                                          \
            return RTM_ECUDA;                                                                      \
        }                                                                                          \
    } while (0)

static inline long long rup(long long v, long long m) { return (v + m - 1) / m * m; }

// Opt a kernel in to the largest dynamic shared memory the device allows (its static shared memory counts against the
// same limit).  The attribute belongs to the function on a device and is shared by all contexts and threads, which is why
// it is never set to one context's own need.
static cudaError_t optin_max_smem(const void *fn, int device) {
    int smem_max = 0;
    cudaError_t e = cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, device);
    if (e != cudaSuccess) return e;
    cudaFuncAttributes fa;
    if ((e = cudaFuncGetAttributes(&fa, fn)) != cudaSuccess) return e;
    return cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max - (int)fa.sharedSizeBytes);
}

// Every entry point runs on the device that owns the context's workspace, whatever device is current in the calling
// thread; the previous device is restored on return.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

// pinned host staging for one set of geometry tables, guarded by an event so that a later call does
// not overwrite it while an earlier upload is still in flight
struct HostTables {
    int *row_start = nullptr;
    InjEntry *ent = nullptr;
    int *smp_idx = nullptr;
    float *smp_w = nullptr;
    cudaEvent_t done = nullptr;
    bool pending = false;
};

struct rtm_ctx {
    rtm_config cfg;
    int device;             // the device d_workspace lives on
    Layout L;
    char *ws;
    size_t ws_bytes;
    int nf;                 // 1 acoustic, 2 TTI
    float *fld[2][3];       // [field][u_a, u_b, du]
    float *fields_base;
    size_t fields_bytes;
    float *K2, *epsh, *delh, *cs, *sn;
    float *cp, *sp, *F[6];   // 3D TTI
    float *dampx, *dampy, *dampz;
    float *k1x, *k1y, *k1z;
    float *Uz, *Vz, *Zf, *Za, *hist;
    int zr, T, rx;
    int tti_tx;   // 2D TTI: rows per tile of tti_step_kernel, 16 (256 threads) or 32 (512 threads; time-blocked probing only)
    long long pNu;   // floats per history slot and per group of planes of one probe: Nu x probed fields
    int rp;   // probe planes per compressed array: r, or 2 r when p and r are probed apart (probe_fields = 2)
    int *row_start;
    InjEntry *ent;
    int *smp_idx;
    float *smp_w;
    int *offs;
    unsigned long long *dbg_ts;
    // resident 2D kernel (acoustic2d_resident.cuh): slab decomposition, exchange buffer, step counters
    struct ResPlan { int nb, groups; size_t smem; } res[2];   // [0] one cluster + DSMEM, [1] exchange through L2; nb = 0: not available
    float *xbuf;
    unsigned *flags;
    int *res_err;
    unsigned res_ep;          // value of the step counters after the last resident launch
    int opt_resident;         // option "resident": 0 never, 1 (default) the cluster mode when the grid fits one, 2 also the L2-exchange mode
    void *tmaps;            // 4 CUtensorMaps of the 3D streaming kernel (u ping, u pong, K2, du), device memory
    long long nrows;
    bool have_model, have_probes, have_U, have_V;
    HostTables ht[2];       // [0] forward call, [1] adjoint call
    int *h_offs;
    cudaEvent_t offs_done;
    bool offs_pending;
    std::vector<int> snap_steps;
    float *snap_out;
    long long launches;
    int opt_time, opt_pdl, opt_dbg;
    static const int kEvRing = 64;
    cudaEvent_t ev[2][kEvRing][2];   // [pass kind][ring slot][begin, end]: the last kEvRing timed passes of each kind
    long long ev_count[2];           // timed passes recorded so far
};

static int pick_rx(rtm_ctx *c);
static int make_tmaps(rtm_ctx *c);
static int plan_resident(rtm_ctx *c);
static int create_on_device(rtm_ctx *c, const rtm_config *cfg, void *d_workspace, size_t bytes);
static size_t stream_smem(const rtm_ctx *c, int rx);
static long long stream_blocks(const rtm_ctx *c, int rx);
static int tm_of(int T);

static bool valid_cfg(const rtm_config *c) {
    if (!c) return false;
    if (c->ndim != 2 && c->ndim != 3) return false;
    for (int a = 0; a < c->ndim; a++)
        if (c->n[a] < 1 || c->n[a] > (1 << 14)) return false;
    if (!(c->h > 0.f) || !std::isfinite(c->h)) return false;
    if (c->nb < 0 || c->nb > 1024) return false;
    if (c->physics != 0 && c->physics != 1) return false;
    if (c->nt < 1 || c->r < 1 || c->r > 256 || c->max_pts < 1) return false;
    // time blocks of up to 16 steps; the acoustic streaming kernels have the registers for 32 history values per
    // flush-role thread, the TTI kernel (64 registers) has not
    if (c->probe_block < 0 || c->probe_block > (c->physics == 0 ? 32 : 16)) return false;
    if (c->probe_block > 16 && c->r > 128) return false;   // staging of the 32 Z rows in the final flush kernel
    // four compressed arrays for the TTI gradient (reading C29): TTI only
    if (c->probe_fields != 0 && c->probe_fields != 1 && c->probe_fields != 2) return false;
    if (c->probe_fields == 2 && c->physics != 1) return false;
    return true;
}

static void make_layout(const rtm_config *c, Layout *L) {
    memset(L, 0, sizeof *L);
    L->nd = c->ndim;
    L->nx = c->n[0];
    L->ny = c->ndim == 3 ? c->n[1] : 1;
    L->nz = c->ndim == 3 ? c->n[2] : c->n[1];
    L->nb = c->nb;
    L->nby = c->ndim == 3 ? c->nb : 0;
    L->H = (c->physics == 1 && c->ndim == 2) ? 8 : 4;   // 2D TTI: two chained derivatives inside one tile; 3D TTI: separate kernels
    L->Hy = c->ndim == 3 ? L->H : 0;
    L->Px = L->nx + 2 * c->nb;
    L->Py = L->ny + 2 * L->nby;
    L->Pzc = L->nz + 2 * c->nb;
    L->zs = (4 - c->nb % 4) % 4;          // alignment points in front of the padded grid (K2 = 0 there)
    L->nbz = c->nb + L->zs;
    L->Pz = L->Pzc + L->zs;
    L->pz = (int)rup(L->Pz + 2 * L->H + 4, 32);
    L->sy = L->pz;
    L->sx = (long long)(L->Py + 2 * L->Hy) * L->pz;
    L->org = (long long)L->H * L->sx + (long long)L->Hy * L->sy + L->H;
    L->fsize = (long long)(L->Px + 2 * L->H) * L->sx + 64;
    L->upz = (int)rup(L->nz, 32);
    L->Nu = (long long)L->nx * L->ny * L->upz;
}

// workspace carving: returns total bytes; fills pointers when ctx != NULL
static size_t carve(const rtm_config *c, const Layout &L, rtm_ctx *ctx) {
    size_t off = 0;
    auto take = [&](size_t bytes) {
        size_t o = off;
        off += (size_t)rup((long long)bytes, 256);
        return o;
    };
    const int nf = c->physics == 1 ? 2 : 1;
    const size_t fb = (size_t)L.fsize * 4;
    size_t o_fields = off;
    size_t o_f[2][3];
    for (int f = 0; f < nf; f++)
        for (int k = 0; k < 3; k++) o_f[f][k] = take(fb);
    size_t fields_bytes = off - o_fields;
    size_t o_K2 = take(fb), o_e = 0, o_d = 0, o_c = 0, o_s = 0;
    if (nf == 2) { o_e = take(fb); o_d = take(fb); o_c = take(fb); o_s = take(fb); }
    const bool tti3 = nf == 2 && c->ndim == 3;
    size_t o_cp = 0, o_sp = 0, o_F[6] = {0, 0, 0, 0, 0, 0};
    if (tti3) { o_cp = take(fb); o_sp = take(fb); for (int k = 0; k < 6; k++) o_F[k] = take(fb); }
    size_t o_dx = take((size_t)(L.Px + 32) * 4), o_dy = take((size_t)(L.Py + 8) * 4), o_dz = take((size_t)(L.Pz + 8) * 4);
    size_t o_kx = take((size_t)(L.Px + 32) * 4), o_ky = take((size_t)(L.Py + 8) * 4), o_kz = take((size_t)(L.Pz + 8) * 4);
    const int rp = c->probe_fields == 2 ? 2 * c->r : c->r;
    size_t pb = (size_t)rp * (size_t)L.Nu * 4;
    size_t o_U = take(pb), o_V = take(pb);
    const int T = c->probe_block > 1 ? c->probe_block : 0;
    size_t o_H = take(2 * (size_t)T * (size_t)(rp / c->r) * (size_t)L.Nu * 4);   // double-buffered history ring (per probed field)
    const int zr = (int)rup(c->r, 8);
    size_t zb = (size_t)c->nt * zr * 4;
    size_t o_Zf = take(zb), o_Za = take(zb);
    const long long nrows = (long long)L.Px * L.Py;
    const int nc = 1 << c->ndim;
    size_t o_rs = take((size_t)(nrows + 1) * 4);
    size_t o_en = take((size_t)c->max_pts * nc * sizeof(InjEntry));
    size_t o_si = take((size_t)c->max_pts * nc * 4), o_sw = take((size_t)c->max_pts * nc * 4);
    size_t o_of = take(5 * 4096 * 4);   // offsets / (ih, hx, hy) triples, then 512 run records of the tiled xy gather
    size_t o_dbg = take(1024 * 8 * 8);
    size_t o_tm = take(4 * 128);
    // resident 2D kernel: step counters (one per SM-slab, 128 bytes apart), error word, exchange buffer [2][NB][8][4 nq]
    const bool res2d = c->ndim == 2 && c->physics == 0 && T > 0;
    size_t o_fl = take(res2d ? 256 * 128 + 256 : 0);
    size_t o_xb = take(res2d ? (size_t)2 * 256 * 8 * (size_t)(L.Pz + 4) * 4 : 0);
    if (ctx) {
        char *b = ctx->ws;
        ctx->nf = nf;
        for (int f = 0; f < 2; f++)
            for (int k = 0; k < 3; k++) ctx->fld[f][k] = f < nf ? (float *)(b + o_f[f][k]) : nullptr;
        ctx->fields_base = (float *)(b + o_fields);
        ctx->fields_bytes = fields_bytes;
        ctx->K2 = (float *)(b + o_K2);
        ctx->epsh = nf == 2 ? (float *)(b + o_e) : nullptr;
        ctx->delh = nf == 2 ? (float *)(b + o_d) : nullptr;
        ctx->cs = nf == 2 ? (float *)(b + o_c) : nullptr;
        ctx->sn = nf == 2 ? (float *)(b + o_s) : nullptr;
        ctx->cp = tti3 ? (float *)(b + o_cp) : nullptr;
        ctx->sp = tti3 ? (float *)(b + o_sp) : nullptr;
        for (int k = 0; k < 6; k++) ctx->F[k] = tti3 ? (float *)(b + o_F[k]) : nullptr;
        ctx->dampx = (float *)(b + o_dx);
        ctx->dampy = (float *)(b + o_dy);
        ctx->dampz = (float *)(b + o_dz);
        ctx->k1x = (float *)(b + o_kx);
        ctx->k1y = (float *)(b + o_ky);
        ctx->k1z = (float *)(b + o_kz);
        ctx->Uz = (float *)(b + o_U);
        ctx->Vz = (float *)(b + o_V);
        ctx->hist = T ? (float *)(b + o_H) : nullptr;
        ctx->T = T;
        ctx->Zf = (float *)(b + o_Zf);
        ctx->Za = (float *)(b + o_Za);
        ctx->zr = zr;
        ctx->rp = rp;
        ctx->pNu = (long long)(rp / c->r) * L.Nu;
        ctx->row_start = (int *)(b + o_rs);
        ctx->ent = (InjEntry *)(b + o_en);
        ctx->smp_idx = (int *)(b + o_si);
        ctx->smp_w = (float *)(b + o_sw);
        ctx->offs = (int *)(b + o_of);
        ctx->dbg_ts = (unsigned long long *)(b + o_dbg);
        ctx->tmaps = b + o_tm;
        ctx->flags = res2d ? (unsigned *)(b + o_fl) : nullptr;
        ctx->res_err = res2d ? (int *)(b + o_fl + 256 * 128) : nullptr;
        ctx->xbuf = res2d ? (float *)(b + o_xb) : nullptr;
        ctx->nrows = nrows;
    }
    return off;
}

extern "C" size_t rtm_workspace_bytes(const rtm_config *cfg) {
    if (!valid_cfg(cfg)) return 0;
    Layout L;
    make_layout(cfg, &L);
    if (L.fsize >= (1LL << 31)) return 0;   // sample tables hold 32-bit offsets
    return carve(cfg, L, nullptr);
}

extern "C" int rtm_create(const rtm_config *cfg, void *d_workspace, size_t bytes, rtm_ctx **out) {
    if (!out) return RTM_EINVAL;
    *out = nullptr;
    size_t need = rtm_workspace_bytes(cfg);
    if (need == 0 || !d_workspace || ((uintptr_t)d_workspace & 255)) return RTM_EINVAL;
    if (bytes < need) return RTM_ENOMEM;
    cudaPointerAttributes pat;
    if (cudaPointerGetAttributes(&pat, d_workspace) != cudaSuccess) { cudaGetLastError(); return RTM_EINVAL; }
    if (pat.type != cudaMemoryTypeDevice && pat.type != cudaMemoryTypeManaged) return RTM_EINVAL;
    rtm_ctx *c = new (std::nothrow) rtm_ctx();
    if (!c) return RTM_ENOMEM;
    c->device = pat.device;
    DeviceGuard guard(c->device);   // events, pinned tables and the occupancy query belong to the workspace's device
    int rc = create_on_device(c, cfg, d_workspace, bytes);
    if (rc) { rtm_destroy(c); return rc; }   // rtm_ctx() value-initialises its pointers: a partial context is safe to destroy
    *out = c;
    return RTM_OK;
}

static int create_on_device(rtm_ctx *c, const rtm_config *cfg, void *d_workspace, size_t bytes) {
    c->cfg = *cfg;
    make_layout(cfg, &c->L);
    c->ws = (char *)d_workspace;
    c->ws_bytes = bytes;
    carve(cfg, c->L, c);
    c->have_model = c->have_probes = c->have_U = c->have_V = false;
    c->snap_out = nullptr;
    c->launches = 0;
    c->opt_time = 0;
    c->opt_pdl = 1;
    c->opt_dbg = 0;
    c->rx = (cfg->ndim == 2 && cfg->physics == 0 && c->T > 0) ? pick_rx(c) : 0;
    c->tti_tx = (cfg->ndim == 2 && cfg->physics == 1 && tm_of(c->T) == 16) ? 32 : 16;
    c->ev_count[0] = c->ev_count[1] = 0;
    for (int i = 0; i < 2; i++)
        for (int s = 0; s < rtm_ctx::kEvRing; s++)
            for (int j = 0; j < 2; j++) CU(cudaEventCreate(&c->ev[i][s][j]));
    c->offs_pending = false;
    const int nc = 1 << cfg->ndim;
    for (int t = 0; t < 2; t++) {
        HostTables &h = c->ht[t];
        CU(cudaMallocHost(&h.row_start, (size_t)(c->nrows + 1) * 4));
        CU(cudaMallocHost(&h.ent, (size_t)cfg->max_pts * nc * sizeof(InjEntry)));
        CU(cudaMallocHost(&h.smp_idx, (size_t)cfg->max_pts * nc * 4));
        CU(cudaMallocHost(&h.smp_w, (size_t)cfg->max_pts * nc * 4));
        CU(cudaEventCreateWithFlags(&h.done, cudaEventDisableTiming));
    }
    CU(cudaMallocHost(&c->h_offs, 5 * 4096 * 4));
    CU(cudaEventCreateWithFlags(&c->offs_done, cudaEventDisableTiming));
    if (cfg->ndim == 3 && cfg->physics == 0 && c->T > 0) return make_tmaps(c);
    c->opt_resident = 1;
    c->res_ep = 0;
    if (cfg->ndim == 2 && cfg->physics == 0 && c->T > 0) return plan_resident(c);
    return RTM_OK;
}

extern "C" void rtm_destroy(rtm_ctx *c) {
    if (!c) return;
    DeviceGuard guard(c->device);
    for (int t = 0; t < 2; t++) {
        HostTables &h = c->ht[t];
        if (h.done) { cudaEventSynchronize(h.done); cudaEventDestroy(h.done); }
        cudaFreeHost(h.row_start); cudaFreeHost(h.ent); cudaFreeHost(h.smp_idx); cudaFreeHost(h.smp_w);
    }
    if (c->offs_done) { cudaEventSynchronize(c->offs_done); cudaEventDestroy(c->offs_done); }
    cudaFreeHost(c->h_offs);
    for (int i = 0; i < 2; i++)
        for (int s = 0; s < rtm_ctx::kEvRing; s++)
            for (int j = 0; j < 2; j++) if (c->ev[i][s][j]) cudaEventDestroy(c->ev[i][s][j]);
    delete c;
}

// ---- O1: coefficients on the host (fp64, one rounding to fp32) ---------------------------------
static int coeffs_host_impl(const rtm_config *cfg, const float *h_vp, const float *h_eps, const float *h_delta,
                            const float *h_theta, const float *h_phi, float *h_K2, float *h_epsh, float *h_delh,
                            float *h_cos, float *h_sin, float *h_cosp, float *h_sinp, float *h_damp1d) {
    if (!valid_cfg(cfg) || !h_vp || !h_K2 || !h_damp1d) return RTM_EINVAL;
    if (cfg->physics == 1 && cfg->ndim == 3 && (!h_phi || !h_cosp || !h_sinp)) return RTM_EINVAL;   // 3D TTI needs the azimuth
    if (!(cfg->dt > 0.0) || !std::isfinite(cfg->dt)) return RTM_EINVAL;   // K2 and the damping tables would be 0 or NaN
    const bool tti = cfg->physics == 1;
    if (tti && (!h_eps || !h_delta || !h_theta || !h_epsh || !h_delh || !h_cos || !h_sin)) return RTM_EINVAL;
    Layout L;
    make_layout(cfg, &L);
    const long long N = (long long)L.nx * L.ny * L.nz;
    const double h = (double)cfg->h, dt = cfg->dt;
    const int nb = cfg->nb;
    double vmax = 0.0;
    for (long long i = 0; i < N; i++) vmax = std::max(vmax, (double)h_vp[i]);
    const double sigma_max = nb > 0 ? vmax * std::log(1000.0) / ((double)nb * h) : 0.0;
    // per-axis profiles sigma_a(i) dt; the dummy y axis of a 2D grid contributes nothing
    const int P[3] = {L.Px, L.Py, L.Pzc};
    const int lay[3] = {nb, L.nby, nb};
    std::vector<double> prof[3];
    float *tab = h_damp1d;
    for (int a = 0; a < 3; a++) {
        prof[a].assign(P[a], 0.0);
        if (cfg->ndim == 2 && a == 1) continue;
        for (int i = 0; i < P[a]; i++) {
            const int depth = std::max(0, std::max(nb - i, i - (P[a] - 1 - nb)));
            const double s = nb > 0 ? (double)depth / (double)nb : 0.0;
            const double phi = s - std::sin(2.0 * M_PI * s) / (2.0 * M_PI);
            prof[a][i] = sigma_max * phi * dt;
            tab[i] = (float)prof[a][i];
        }
        tab += P[a];
    }
    // Edge replication into the layer as per-axis index maps (physical index of every padded index), then one sweep over
    // the padded grid in canonical order.  sigma dt = (x part + y part) + z part, in that association: it is rounded
    // once to fp32 through K2 and must give the same bits on every implementation of O1.
    std::vector<int> src_of[3];
    const int nn[3] = {L.nx, L.ny, L.nz};
    for (int a = 0; a < 3; a++) {
        src_of[a].resize(P[a]);
        for (int j = 0; j < P[a]; j++) src_of[a][j] = std::min(std::max(j - lay[a], 0), nn[a] - 1);
    }
    long long d = 0;
    for (int jx = 0; jx < L.Px; jx++) {
        const long long sx_ = (long long)src_of[0][jx] * L.ny;
        for (int jy = 0; jy < L.Py; jy++) {
            const long long sxy = (sx_ + src_of[1][jy]) * L.nz;
            const double pxy = prof[0][jx] + prof[1][jy];
            for (int jz = 0; jz < L.Pzc; jz++, d++) {
                const long long s = sxy + src_of[2][jz];
                const double c = h_vp[s];
                h_K2[d] = (float)(c * c * dt * dt / (h * h * (1.0 + (pxy + prof[2][jz]))));
                if (!tti) continue;
                const double e = h_eps[s];
                h_epsh[d] = (float)(1.0 + 2.0 * e);
                h_delh[d] = (float)std::sqrt(1.0 + 2.0 * std::min((double)h_delta[s], e));
                h_cos[d] = (float)std::cos((double)h_theta[s]);
                h_sin[d] = (float)std::sin((double)h_theta[s]);
                if (h_phi) {
                    h_cosp[d] = (float)std::cos((double)h_phi[s]);
                    h_sinp[d] = (float)std::sin((double)h_phi[s]);
                }
            }
        }
    }
    return RTM_OK;
}
extern "C" int rtm_coeffs_host(const rtm_config *cfg, const float *h_vp, const float *h_eps, const float *h_delta,
                               const float *h_theta, float *h_K2, float *h_epsh, float *h_delh, float *h_cos,
                               float *h_sin, float *h_damp1d) {
    return coeffs_host_impl(cfg, h_vp, h_eps, h_delta, h_theta, nullptr, h_K2, h_epsh, h_delh, h_cos, h_sin, nullptr, nullptr, h_damp1d);
}
extern "C" int rtm_coeffs_host3(const rtm_config *cfg, const float *h_vp, const float *h_eps, const float *h_delta,
                                const float *h_theta, const float *h_phi, float *h_K2, float *h_epsh, float *h_delh,
                                float *h_cos, float *h_sin, float *h_cosp, float *h_sinp, float *h_damp1d) {
    if (!cfg || cfg->physics != 1 || cfg->ndim != 3) return RTM_EINVAL;
    return coeffs_host_impl(cfg, h_vp, h_eps, h_delta, h_theta, h_phi, h_K2, h_epsh, h_delh, h_cos, h_sin, h_cosp, h_sinp, h_damp1d);
}

// ---- reading C4: second time difference moved from the wavefield onto the probes (host, fp64) ------------
extern "C" int rtm_probes_dtt_host(int nt, int r, double dt, const float *h_Z, float *h_Zdd) {
    if (nt < 1 || r < 1 || !(dt > 0.0) || !h_Z || !h_Zdd || h_Z == h_Zdd) return RTM_EINVAL;
    const double s = 1.0 / (dt * dt);
    for (int n = 0; n < nt; n++)
        for (int k = 0; k < r; k++) {
            const double z0 = h_Z[(size_t)n * r + k];
            const double z1 = n + 1 < nt ? (double)h_Z[(size_t)(n + 1) * r + k] : 0.0;
            const double z2 = n + 2 < nt ? (double)h_Z[(size_t)(n + 2) * r + k] : 0.0;
            h_Zdd[(size_t)n * r + k] = (float)(((z0 - 2.0 * z1) + z2) * s);
        }
    return RTM_OK;
}

// ---- reading C3: range-finder probes [Q, ~] = qr(A Z), A = D D^T (host, fp64) -------------------
// Y = D (D^T Z) without forming the nt x nt matrix, then Gram-Schmidt with one re-orthogonalisation pass per column
// (the "twice is enough" variant: orthogonal to rounding for any Y that is not numerically rank-deficient).
// Normalising by a positive norm gives the thin QR with diag(R) > 0, the unique one.
extern "C" int rtm_probes_qr_host(int nt, int nrec, int r, const float *h_D, const float *h_Z, float *h_Q) {
    if (nt < 1 || nrec < 1 || r < 1 || r > nt || !h_D || !h_Z || !h_Q || h_Z == h_Q) return RTM_EINVAL;
    std::vector<double> W((size_t)nrec * r, 0.0), Y((size_t)r * nt, 0.0);   // W = D^T Z [nrec][r]; Y column-major [r][nt]
    for (int n = 0; n < nt; n++)
        for (int j = 0; j < nrec; j++) {
            const double d = h_D[(size_t)n * nrec + j];
            for (int k = 0; k < r; k++) W[(size_t)j * r + k] += d * (double)h_Z[(size_t)n * r + k];
        }
    for (int n = 0; n < nt; n++)
        for (int j = 0; j < nrec; j++) {
            const double d = h_D[(size_t)n * nrec + j];
            for (int k = 0; k < r; k++) Y[(size_t)k * nt + n] += d * W[(size_t)j * r + k];
        }
    for (int k = 0; k < r; k++) {
        double *y = &Y[(size_t)k * nt];
        double n0 = 0.0;
        for (int n = 0; n < nt; n++) n0 += y[n] * y[n];
        for (int pass = 0; pass < 2; pass++)
            for (int i = 0; i < k; i++) {
                const double *q = &Y[(size_t)i * nt];
                double dot = 0.0;
                for (int n = 0; n < nt; n++) dot += q[n] * y[n];
                for (int n = 0; n < nt; n++) y[n] -= dot * q[n];
            }
        double n1 = 0.0;
        for (int n = 0; n < nt; n++) n1 += y[n] * y[n];
        if (!(n1 > 1e-24 * n0) || !(n0 > 0.0)) return RTM_EINVAL;   // A Z is numerically rank-deficient (r > rank D)
        const double inv = 1.0 / std::sqrt(n1);
        for (int n = 0; n < nt; n++) y[n] *= inv;
    }
    for (int n = 0; n < nt; n++)
        for (int k = 0; k < r; k++) h_Q[(size_t)n * r + k] = (float)Y[(size_t)k * nt + n];
    return RTM_OK;
}

static int launch_pack(rtm_ctx *c, const float *src, float *dst, cudaStream_t st) {
    const long long Np = (long long)c->L.Px * c->L.Py * c->L.Pzc;
    pack_field_kernel<<<(unsigned)((Np + 255) / 256), 256, 0, st>>>(c->L, src, dst);
    c->launches++;
    CU(cudaGetLastError());
    return RTM_OK;
}

static int set_model_impl(rtm_ctx *c, const float *d_K2, const float *d_epsh, const float *d_delh, const float *d_cos,
                          const float *d_sin, const float *d_cosp, const float *d_sinp, const float *h_damp1d, void *stream) {
    if (!c || !d_K2 || !h_damp1d) return RTM_EINVAL;
    DeviceGuard guard(c->device);
    const bool tti = c->cfg.physics == 1;
    if (tti && (!d_epsh || !d_delh || !d_cos || !d_sin)) return RTM_EINVAL;
    if (tti && c->cfg.ndim == 3 && (!d_cosp || !d_sinp)) return RTM_EINVAL;   // 3D TTI: use rtm_set_model3
    cudaStream_t st = (cudaStream_t)stream;
    const Layout &L = c->L;
    // zero everything up to the probe planes once (halo of fields and coefficients stays zero)
    CU(cudaMemsetAsync(c->ws, 0, (size_t)((char *)c->Uz - c->ws), st));
    int rc;
    if ((rc = launch_pack(c, d_K2, c->K2, st))) return rc;
    if (tti) {
        if ((rc = launch_pack(c, d_epsh, c->epsh, st))) return rc;
        if ((rc = launch_pack(c, d_delh, c->delh, st))) return rc;
        if ((rc = launch_pack(c, d_cos, c->cs, st))) return rc;
        if ((rc = launch_pack(c, d_sin, c->sn, st))) return rc;
        if (c->cfg.ndim == 3) {
            if ((rc = launch_pack(c, d_cosp, c->cp, st))) return rc;
            if ((rc = launch_pack(c, d_sinp, c->sp, st))) return rc;
        }
    }
    // small tables: pageable source, the copy is staged before the call returns
    const float *t = h_damp1d;
    CU(cudaMemcpyAsync(c->dampx, t, (size_t)L.Px * 4, cudaMemcpyHostToDevice, st));
    t += L.Px;
    if (c->cfg.ndim == 3) {
        CU(cudaMemcpyAsync(c->dampy, t, (size_t)L.Py * 4, cudaMemcpyHostToDevice, st));
        t += L.Py;
    }
    CU(cudaMemcpyAsync(c->dampz + L.zs, t, (size_t)L.Pzc * 4, cudaMemcpyHostToDevice, st));   // the zs alignment points keep 0
    // per-axis K1 tables, computed on the device with the same division the kernels use at layer corners
    k1_table_kernel<<<(L.Px + 32 + 255) / 256, 256, 0, st>>>(c->dampx, c->k1x, L.Px + 32);
    k1_table_kernel<<<(L.Py + 8 + 255) / 256, 256, 0, st>>>(c->dampy, c->k1y, L.Py + 8);
    k1_table_kernel<<<(L.Pz + 8 + 255) / 256, 256, 0, st>>>(c->dampz, c->k1z, L.Pz + 8);
    c->launches += 3;
    CU(cudaGetLastError());
    c->have_model = true;
    c->have_U = c->have_V = false;
    return RTM_OK;
}

extern "C" int rtm_set_model(rtm_ctx *c, const float *d_K2, const float *d_epsh, const float *d_delh,
                             const float *d_cos, const float *d_sin, const float *h_damp1d, void *stream) {
    return set_model_impl(c, d_K2, d_epsh, d_delh, d_cos, d_sin, nullptr, nullptr, h_damp1d, stream);
}
extern "C" int rtm_set_model3(rtm_ctx *c, const float *d_K2, const float *d_epsh, const float *d_delh, const float *d_cos,
                              const float *d_sin, const float *d_cosp, const float *d_sinp, const float *h_damp1d, void *stream) {
    if (!c || c->cfg.physics != 1 || c->cfg.ndim != 3) return RTM_EINVAL;
    return set_model_impl(c, d_K2, d_epsh, d_delh, d_cos, d_sin, d_cosp, d_sinp, h_damp1d, stream);
}

extern "C" int rtm_set_probes(rtm_ctx *c, const float *d_Zf, const float *d_Za, void *stream) {
    if (!c || !d_Zf || !d_Za) return RTM_EINVAL;
    DeviceGuard guard(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    const long long tot = (long long)c->cfg.nt * c->zr;
    pack_probes_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(c->cfg.nt, c->cfg.r, c->zr, d_Zf, c->Zf);
    pack_probes_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(c->cfg.nt, c->cfg.r, c->zr, d_Za, c->Za);
    c->launches += 2;
    CU(cudaGetLastError());
    c->have_probes = true;
    return RTM_OK;
}

// ---- geometry (reading C9): multilinear corners and weights -------------------------------------
struct Corner { int jx, jy, jz; float w; };

// returns the number of corners (2^d) or -1 if the position is outside [0,(n_a-1)h]
static int corners_of(const rtm_config &cfg, const Layout &L, const float *xyz, Corner *out) {
    const int nn[3] = {L.nx, L.ny, L.nz};
    int base[3] = {0, 0, 0};
    double frac[3] = {0.0, 0.0, 0.0};
    int k = 0;
    for (int a = 0; a < 3; a++) {
        if (cfg.ndim == 2 && a == 1) continue;
        const double f = (double)xyz[k++] / (double)cfg.h;
        if (!(f >= 0.0) || f > (double)(nn[a] - 1)) return -1;
        int i = (int)std::floor(f);
        i = std::max(0, std::min(i, nn[a] - 2));
        base[a] = i;
        frac[a] = f - (double)i;
    }
    int cnt = 0;
    for (int bx = 0; bx < 2; bx++)
        for (int by = 0; by < 2; by++)
            for (int bz = 0; bz < 2; bz++) {
                if (cfg.ndim == 2 && by) continue;
                Corner &co = out[cnt++];
                if ((bx && nn[0] == 1) || (by && nn[1] == 1) || (bz && nn[2] == 1)) { co = {0, 0, 0, 0.f}; continue; }
                double w = bx ? frac[0] : 1.0 - frac[0];
                if (cfg.ndim == 3) w *= by ? frac[1] : 1.0 - frac[1];
                w *= bz ? frac[2] : 1.0 - frac[2];
                co.jx = base[0] + bx + L.nb;
                co.jy = base[1] + by + L.nby;
                co.jz = base[2] + bz + L.nbz;
                co.w = (float)w;
            }
    return cnt;
}

// slab of the resident 2D kernel that owns padded row jx (the first rrem slabs have one row more)
static int slab_of_row(const rtm_ctx *c, int nb, int jx) {
    const int rbase = c->L.Px / nb, rrem = c->L.Px % nb;
    const int big = rrem * (rbase + 1);
    return jx < big ? jx / (rbase + 1) : rrem + (jx - big) / rbase;
}

struct PassGeom {
    int ninj, nsmp, nc;
    int bx0, bx1, by0, by1, bz0, bz1;
    bool res_ok[2];   // the resident 2D kernel's per-slab tables (injection groups, sampled points) can hold this geometry, per mode
};

// Build injection (row-CSR) and sampling tables on the host and upload them.
static int build_geometry(rtm_ctx *c, int slot, int ninj, const float *inj_xyz, int nsmp, const float *smp_xyz,
                          PassGeom *g, cudaStream_t st) {
    const rtm_config &cfg = c->cfg;
    const Layout &L = c->L;
    const int nd = cfg.ndim, nc = 1 << nd;
    HostTables &h = c->ht[slot];
    if (h.pending) { CU(cudaEventSynchronize(h.done)); h.pending = false; }
    g->ninj = ninj; g->nsmp = nsmp; g->nc = nc;
    g->bx0 = g->by0 = g->bz0 = 1 << 30;
    g->bx1 = g->by1 = g->bz1 = -1;
    struct Tmp { long long row; int jz, id; float w; };
    std::vector<Tmp> tmp;
    tmp.reserve((size_t)ninj * nc);
    Corner co[8];
    for (int s = 0; s < ninj; s++) {
        if (corners_of(cfg, L, inj_xyz + (size_t)s * nd, co) < 0) return RTM_EINVAL;
        for (int k = 0; k < nc; k++) {
            if (co[k].w == 0.f) continue;
            tmp.push_back({(long long)co[k].jx * L.Py + co[k].jy, co[k].jz, s, co[k].w});
            g->bx0 = std::min(g->bx0, co[k].jx); g->bx1 = std::max(g->bx1, co[k].jx);
            g->by0 = std::min(g->by0, co[k].jy); g->by1 = std::max(g->by1, co[k].jy);
            g->bz0 = std::min(g->bz0, co[k].jz); g->bz1 = std::max(g->bz1, co[k].jz);
        }
    }
    std::sort(tmp.begin(), tmp.end(), [](const Tmp &a, const Tmp &b) {
        if (a.row != b.row) return a.row < b.row;
        if (a.jz != b.jz) return a.jz < b.jz;
        return a.id < b.id;
    });
    std::fill(h.row_start, h.row_start + c->nrows + 1, 0);
    for (const Tmp &t : tmp) h.row_start[t.row + 1]++;
    for (long long i = 0; i < c->nrows; i++) h.row_start[i + 1] += h.row_start[i];
    for (size_t i = 0; i < tmp.size(); i++) h.ent[i] = {tmp[i].jz, tmp[i].id, tmp[i].w, 0};
    // resident 2D kernel: do the per-slab tables hold this geometry?  (injection groups = distinct (row, quad) pairs)
    std::vector<int> per_slab[2];
    for (int m = 0; m < 2; m++) {
        g->res_ok[m] = c->res[m].nb > 0;
        per_slab[m].assign(std::max(1, c->res[m].nb), 0);
        if (!g->res_ok[m]) continue;
        long long lrow = -1; int lq = -1;
        std::vector<int> ents(per_slab[m].size(), 0);
        for (const Tmp &t : tmp) {
            const int sl = slab_of_row(c, c->res[m].nb, (int)t.row);
            ents[sl]++;
            if (t.row != lrow || (t.jz >> 2) != lq) { per_slab[m][sl]++; lrow = t.row; lq = t.jz >> 2; }
        }
        for (size_t i = 0; i < ents.size(); i++) g->res_ok[m] = g->res_ok[m] && per_slab[m][i] <= RS_MAXG && ents[i] <= RS_MAXE;
        std::fill(per_slab[m].begin(), per_slab[m].end(), 0);
    }
    for (int s = 0; s < nsmp; s++) {
        if (corners_of(cfg, L, smp_xyz + (size_t)s * nd, co) < 0) return RTM_EINVAL;
        for (int k = 0; k < nc; k++) {
            h.smp_idx[(size_t)s * nc + k] = (int)(L.org + co[k].jx * L.sx + co[k].jy * L.sy + co[k].jz);
            h.smp_w[(size_t)s * nc + k] = co[k].w;
        }
        for (int m = 0; m < 2; m++)
            if (g->res_ok[m]) g->res_ok[m] = ++per_slab[m][slab_of_row(c, c->res[m].nb, co[0].jx)] <= RS_MAXS;
    }
    CU(cudaMemcpyAsync(c->row_start, h.row_start, (size_t)(c->nrows + 1) * 4, cudaMemcpyHostToDevice, st));
    if (!tmp.empty())
        CU(cudaMemcpyAsync(c->ent, h.ent, tmp.size() * sizeof(InjEntry), cudaMemcpyHostToDevice, st));
    if (nsmp > 0) {
        CU(cudaMemcpyAsync(c->smp_idx, h.smp_idx, (size_t)nsmp * nc * 4, cudaMemcpyHostToDevice, st));
        CU(cudaMemcpyAsync(c->smp_w, h.smp_w, (size_t)nsmp * nc * 4, cudaMemcpyHostToDevice, st));
    }
    CU(cudaEventRecord(h.done, st));
    h.pending = true;
    return RTM_OK;
}

// ---- tensor maps of the 3D streaming kernel (TMA, acoustic3d_stream.cuh) ---------------------------------------
// A field is a dense [Px + 2H][Py + 2H][pz] array of floats (halo included); the kernel asks for boxes by (z, y, x)
// counted from the first float.  u ping / pong: haloed boxes 136 x 16 x 1; K2, du: 128 x 8 x 1.  Whatever part of a
// box lies outside the array is filled with zeros by the copy engine.
static int make_tmaps(rtm_ctx *c) {
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    CU(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
    if (!fn || qres != cudaDriverEntryPointSuccess) {
        snprintf(g_cuda_err, sizeof g_cuda_err, "cuTensorMapEncodeTiled is not available in this driver");
        return RTM_ECUDA;
    }
    const Layout &L = c->L;
    const cuuint64_t dims[3] = {(cuuint64_t)L.pz, (cuuint64_t)(L.Py + 2 * L.Hy), (cuuint64_t)(L.Px + 2 * L.H)};
    const cuuint64_t strides[2] = {(cuuint64_t)L.sy * 4, (cuuint64_t)L.sx * 4};
    const cuuint32_t ones[3] = {1, 1, 1};
    const cuuint32_t box_u[3] = {(cuuint32_t)S3_PITCH, (cuuint32_t)S3_ROWS, 1}, box_k[3] = {(cuuint32_t)S3_TZ, (cuuint32_t)S3_TY, 1};
    alignas(64) CUtensorMap maps[4];
    static_assert(sizeof(CUtensorMap) == 128, "the kernel addresses the maps at multiples of 128 bytes");
    void *base[4] = {c->fld[0][0], c->fld[0][1], c->K2, c->fld[0][2]};
    for (int i = 0; i < 4; i++) {
        CUresult r = ((encode_fn)fn)(&maps[i], CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, base[i], dims, strides, i < 2 ? box_u : box_k,
                                     ones, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                     CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) {
            snprintf(g_cuda_err, sizeof g_cuda_err, "cuTensorMapEncodeTiled failed with CUresult %d (map %d)", (int)r, i);
            return RTM_ECUDA;
        }
    }
    CU(cudaMemcpy(c->tmaps, maps, sizeof maps, cudaMemcpyHostToDevice));
    return RTM_OK;
}

// ---- resident 2D kernel: plan and launch (acoustic2d_resident.cuh) ----------------------------------------------------
static size_t resident_smem(const Layout &L, int rmax, int mode) {
    const int nq = (L.Pz + 3) / 4, spz = nq * 4 + 8;
    return (size_t)2 * (rmax + 8) * spz * 4 + (size_t)rmax * nq * 16 * (mode == 0 ? 2 : 1) /* du (+ K2 in the cluster mode) */ +
           (size_t)(RS_MAXG + 1) * (16 + sizeof(RsGroup)) + (size_t)RS_MAXE * (sizeof(InjEntry) + 8) +
           (size_t)RS_MAXS * sizeof(RsSample) + (size_t)rmax * nq + 16;
}
// Mode 1 (exchange through L2): one slab per SM, the largest NB <= #SM whose slabs have >= 4 rows (a halo comes from ONE
// neighbour).  Mode 0 (one cluster): the same with NB <= 16 blocks that form one thread-block cluster.  A plan stands if
// the slabs fit the shared memory of an SM and the threads of a block cover the quad columns.
static int plan_resident(rtm_ctx *c) {
    const Layout &L = c->L;
    c->res[0].nb = c->res[1].nb = 0;
    int nsm = 0, smem_max = 0;
    CU(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, c->device));
    CU(cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, c->device));
    const int nq = (L.Pz + 3) / 4;
    for (int m = 0; m < 2; m++) {
        const void *fn = m == 0 ? (const void *)acoustic2d_resident_kernel<true> : (const void *)acoustic2d_resident_kernel<false>;
        for (int cap = m == 0 ? 16 : std::min(nsm, 256); cap >= (m == 0 ? 2 : 1); cap = m == 0 ? cap / 2 : 0) {
            const int nb = std::min(cap, L.Px / 4);
            if (nb < 1 || (m == 0 && nb < 2)) break;
            if (m == 1 ? 2 * nq > RS_THREADS - 32 : nq > RS_THREADS) break;   // mode 1: two sweeping threads per column + the communication warp
            const int rmax = (L.Px + nb - 1) / nb;
            if (rmax > RS_MAXROWS) break;
            const size_t smem = resident_smem(L, rmax, m);
            if (smem + 1024 > (size_t)smem_max) break;
            // the opt-in is a property of the FUNCTION on this device, shared by every context: always the device maximum,
            // never this context's own need (a second, smaller context must not lower it under the first one's feet)
            CU(optin_max_smem(fn, c->device));
            if (m == 0) {
                CU(cudaFuncSetAttribute(fn, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
                cudaLaunchAttribute at[1];
                at[0].id = cudaLaunchAttributeClusterDimension;
                at[0].val.clusterDim.x = (unsigned)nb; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
                cudaLaunchConfig_t lc;
                memset(&lc, 0, sizeof lc);
                lc.gridDim = dim3((unsigned)nb, 1, 1); lc.blockDim = dim3(RS_THREADS, 1, 1); lc.dynamicSmemBytes = smem;
                lc.attrs = at; lc.numAttrs = 1;
                int ncl = 0;
                if (cudaOccupancyMaxActiveClusters(&ncl, fn, &lc) != cudaSuccess || ncl < 1) { cudaGetLastError(); continue; }   // try a smaller cluster
            } else {
                int per_sm = 0;
                CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, acoustic2d_resident_kernel<false>, RS_THREADS, smem));
                if (per_sm < 1) break;
            }
            c->res[m].nb = nb;
            c->res[m].groups = m == 0 ? std::max(1, std::min(L.Px / nb, RS_THREADS / nq)) : 2;
            c->res[m].smem = smem;
            break;
        }
    }
    CU(cudaMemset(c->flags, 0, 256 * 128 + 256));
    return RTM_OK;
}

// nsteps steps starting at time index n0, fields in fld[0][cur] / fld[0][2], history slots hist0, hist0 + pNu, ...
static int launch_resident(rtm_ctx *c, int mode, const StepArgs &a, int adjoint, int n0, int nsteps, int cur, const PassGeom &g,
                           const float *d_inj_val, float *d_smp_out, float *hist0, cudaStream_t st) {
    const Layout &L = c->L;
    ResidentArgs ra;
    memset(&ra, 0, sizeof ra);
    const rtm_ctx::ResPlan &pl = c->res[mode];
    ra.NB = pl.nb;
    ra.rbase = L.Px / pl.nb; ra.rrem = L.Px % pl.nb; ra.rmax = ra.rbase + (ra.rrem ? 1 : 0);
    ra.nq = (L.Pz + 3) / 4; ra.spz = ra.nq * 4 + 8;
    ra.groups = pl.groups;
    ra.nsteps = nsteps; ra.n0 = n0; ra.dir = adjoint ? -1 : 1;
    ra.ninj = g.ninj; ra.inj_base = d_inj_val;
    ra.smp_base = (d_smp_out != nullptr && g.nsmp > 0) ? d_smp_out : nullptr;
    ra.hist0 = hist0;
    ra.u = c->fld[0][cur]; ra.du = c->fld[0][2];
    ra.xbuf = c->xbuf; ra.flags = c->flags; ra.err = c->res_err;
    ra.ep0 = c->res_ep;
    c->res_ep += (unsigned)nsteps;
    cudaLaunchAttribute at[1];
    if (mode == 0) {
        at[0].id = cudaLaunchAttributeClusterDimension;   // one cluster: co-scheduled by construction
        at[0].val.clusterDim.x = (unsigned)pl.nb; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    } else {
        at[0].id = cudaLaunchAttributeCooperative;        // all blocks co-resident, or the launch fails: blocks wait for their neighbours
        at[0].val.cooperative = 1;
    }
    cudaLaunchConfig_t lc;
    memset(&lc, 0, sizeof lc);
    lc.gridDim = dim3((unsigned)pl.nb, 1, 1); lc.blockDim = dim3(RS_THREADS, 1, 1);
    lc.dynamicSmemBytes = pl.smem; lc.stream = st; lc.attrs = at; lc.numAttrs = 1;
    if (mode == 0) CU(cudaLaunchKernelEx(&lc, acoustic2d_resident_kernel<true>, a, ra));
    else CU(cudaLaunchKernelEx(&lc, acoustic2d_resident_kernel<false>, a, ra));
    c->launches++;
    return RTM_OK;
}

// ---- one propagation pass (a1-a6) ---------------------------------------------------------------
static void step_grid(const rtm_ctx *c, dim3 *grid, dim3 *block, size_t *smem) {
    const Layout &L = c->L;
    if (c->cfg.physics == 1 && c->cfg.ndim == 3) {
        *grid = dim3((L.Pz + 127) / 128, (L.Py + 7) / 8, L.Px);
        *block = dim3(32, 8, 1);
        *smem = 0;
    } else if (c->cfg.physics == 1) {
        *grid = dim3((L.Pz + TTI_TZ - 1) / TTI_TZ, (L.Px + c->tti_tx - 1) / c->tti_tx, 1);
        *block = dim3(16, c->tti_tx, 1);
        *smem = std::max<size_t>((size_t)tti_smem(c->tti_tx), (size_t)tm_of(c->T) * c->zr * 4);
    } else if (c->cfg.ndim == 2 && c->T > 0) {
        // streaming kernel: 1-D list of (row chunk, z-quad) tasks, 128 per block; grid.x = blocks,
        // a.gx is overwritten with the quads per row by run_pass
        *grid = dim3((unsigned)stream_blocks(c, c->rx), 1, 1);
        *block = dim3(128, 1, 1);
        *smem = stream_smem(c, c->rx);
    } else if (c->cfg.ndim == 2) {
        *grid = dim3((L.Pz + 127) / 128, (L.Px + 7) / 8, 1);
        *block = dim3(32, 8, 1);
        *smem = 0;
    } else if (c->T > 0) {
        // 2.5D streaming kernel: (y, z) tiles of 8 x 128, chunks of S3_XCH planes along x
        *grid = dim3((L.Pz + S3_TZ - 1) / S3_TZ, (L.Py + S3_TY - 1) / S3_TY, (L.Px + S3_XCH - 1) / S3_XCH);
        *block = dim3(256, 1, 1);
        *smem = std::max<size_t>((size_t)S3_SMEM, (size_t)tm_of(c->T) * c->zr * 4);
    } else {
        *grid = dim3((L.Pz + 127) / 128, (L.Py + 7) / 8, L.Px);
        *block = dim3(32, 8, 1);
        *smem = 0;
    }
}

typedef void (*step_fn)(const StepArgs);
static int tm_of(int T);
// ---- launch shape of the 2D streaming kernel ---------------------------------------------------------------
static const size_t kSmemBudget = 56 * 1024;   // per block: four blocks per SM
static long long stream_blocks(const rtm_ctx *c, int rx) {
    const Layout &L = c->L;
    const long long nq = (L.Pz + 3) / 4, nchunk = (L.Px + rx - 1) / rx;
    return (nq * nchunk + 127) / 128;
}
// dynamic shared memory: injection amounts [RX][128] float4 (stencil role) or the Z rows [TM][zr] (flush role),
// whichever is larger
static size_t stream_smem(const rtm_ctx *c, int rx) {
    const int rxt = rx <= 2 ? 2 : rx <= 4 ? 4 : rx <= 8 ? 8 : 16;
    return std::max<size_t>((size_t)rxt * 128 * 16, (size_t)tm_of(c->T) * c->zr * 4);
}
template <int TM>
static step_fn stream2d_fn(int rx) {
    return rx <= 2 ? acoustic2d_stream_kernel<TM, 2> : rx <= 4 ? acoustic2d_stream_kernel<TM, 4>
         : rx <= 8 ? acoustic2d_stream_kernel<TM, 8> : acoustic2d_stream_kernel<TM, 16>;
}
// Rows per thread of the 2D streaming kernel: the smallest RX in {2,4,8,16} whose launch (stencil + flush blocks) fits
// in two waves of resident blocks; larger problems use 4.
static int pick_rx(rtm_ctx *c) {
    int nsm = 148;
    cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, c->device);
    const int tm = tm_of(c->T);
    // flush-role blocks that share every launch: one float4 of the physical grid per thread, 1/T of it per step
    const long long quads = (long long)c->L.nx * c->L.ny * (c->L.upz / (c->T <= 16 ? 4 : 2));
    const long long fblocks = (quads / std::max(1, c->T - 1) + 127) / 128 + 1;
    const int cand[4] = {2, 4, 8, 16};
    for (int i = 0; i < 4; i++) {
        step_fn f = tm <= 4 ? stream2d_fn<4>(cand[i]) : tm <= 8 ? stream2d_fn<8>(cand[i]) : tm <= 16 ? stream2d_fn<16>(cand[i]) : stream2d_fn<32>(cand[i]);
        int per_sm = 0;
        cudaFuncSetAttribute((const void *)f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBudget);
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, f, 128, stream_smem(c, cand[i])) != cudaSuccess) { cudaGetLastError(); continue; }
        // measured at c1 (1911 x 911, T = 16): RX = 4 (1028 blocks, 1.7 waves) 12.4 us per step, RX = 8 (591 blocks, one
        // wave) 13.5 us, RX = 16 15.9 us: fine-grained blocks balance the stencil and flush roles better than one
        // wave of long-lived ones, as long as the launch stays within two waves
        if (stream_blocks(c, cand[i]) + fblocks <= 2LL * per_sm * nsm) return cand[i];
    }
    return 4;
}

static int tm_of(int T) { return T <= 0 ? 0 : T <= 4 ? 4 : T <= 8 ? 8 : T <= 16 ? 16 : 32; }

template <typename K>
static int launch_ex(rtm_ctx *c, K kernel, const StepArgs &a, unsigned nblocks, dim3 block, size_t smem, cudaStream_t st) {
    // programmatic dependent launch: the grid may become resident while its predecessor drains; the
    // kernels call griddepcontrol.wait before touching memory
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = c->opt_pdl ? 1 : 0;
    cudaLaunchConfig_t lc;
    memset(&lc, 0, sizeof lc);
    lc.gridDim = dim3(nblocks, 1, 1); lc.blockDim = block; lc.dynamicSmemBytes = smem; lc.stream = st;
    lc.attrs = at; lc.numAttrs = 1;
    if (smem > 48 * 1024) {
        // opt in to large dynamic shared memory, once per (device, kernel) and thread: the attribute belongs to the
        // function on a device and is shared by all contexts and threads, so it is always set to the device maximum
        struct Done { int dev; const void *fp; };
        static thread_local std::vector<Done> done;
        const void *fp = (const void *)kernel;
        bool ok = false;
        for (auto &d : done) ok = ok || (d.dev == c->device && d.fp == fp);
        if (!ok) {
            CU(optin_max_smem(fp, c->device));
            done.push_back({c->device, fp});
        }
    }
    CU(cudaLaunchKernelEx(&lc, kernel, a));
    c->launches++;
    return RTM_OK;
}

// the launch grid is 1-D: a.fl_blocks flush-role blocks first, then the gx*gy*gz stencil blocks
static int launch_step(rtm_ctx *c, const StepArgs &a, dim3 grid, dim3 block, size_t smem, cudaStream_t st) {
    const unsigned nb = a.fl_blocks + grid.x * grid.y * grid.z;
    const int tm = tm_of(c->T);
    if (c->cfg.physics == 1 && c->cfg.ndim == 3) {   // mix (adjoint), rotated gradients, divergence + update
        int rc = 0;
        if (a.adjoint && (rc = launch_ex(c, tti3d_mix_kernel, a, nb, block, 0, st))) return rc;
        if ((rc = launch_ex(c, tti3d_grad_kernel, a, nb, block, 0, st))) return rc;
        if (a.two) return tm == 0 ? launch_ex(c, tti3d_step_kernel<0, true>, a, nb, block, 0, st) : launch_ex(c, tti3d_step_kernel<16, true>, a, nb, block, 0, st);
        return tm == 0 ? launch_ex(c, tti3d_step_kernel<0>, a, nb, block, 0, st) : launch_ex(c, tti3d_step_kernel<16>, a, nb, block, 0, st);
    } else if (c->cfg.physics == 1) {
        switch (tm) {
            case 0: return a.two ? launch_ex(c, tti_step_kernel<0, true>, a, nb, block, smem, st)
                                 : launch_ex(c, tti_step_kernel<0>, a, nb, block, smem, st);
            case 4: return a.two ? launch_ex(c, tti_step_kernel<4, true>, a, nb, block, smem, st)
                                 : launch_ex(c, tti_step_kernel<4>, a, nb, block, smem, st);
            case 8: return a.two ? launch_ex(c, tti_step_kernel<8, true>, a, nb, block, smem, st)
                                 : launch_ex(c, tti_step_kernel<8>, a, nb, block, smem, st);
            default:
                if (c->tti_tx == 32) return a.two ? launch_ex(c, tti_step_kernel<16, true, 32>, a, nb, block, smem, st)
                                                  : launch_ex(c, tti_step_kernel<16, false, 32>, a, nb, block, smem, st);
                return a.two ? launch_ex(c, tti_step_kernel<16, true>, a, nb, block, smem, st)
                             : launch_ex(c, tti_step_kernel<16>, a, nb, block, smem, st);
        }
    } else if (c->cfg.ndim == 2) {
        switch (tm) {
            case 0: return launch_ex(c, acoustic_step_kernel<2>, a, nb, block, 0, st);
            case 4: return launch_ex(c, stream2d_fn<4>(c->rx), a, nb, block, smem, st);
            case 8: return launch_ex(c, stream2d_fn<8>(c->rx), a, nb, block, smem, st);
            case 16: return launch_ex(c, stream2d_fn<16>(c->rx), a, nb, block, smem, st);
            default: return launch_ex(c, stream2d_fn<32>(c->rx), a, nb, block, smem, st);
        }
    } else {
        switch (tm) {
            case 0: return launch_ex(c, acoustic_step_kernel<3>, a, nb, block, 0, st);
            case 4: return launch_ex(c, acoustic3d_stream_kernel<4, true>, a, nb, block, smem, st);
            case 8: return launch_ex(c, acoustic3d_stream_kernel<8, true>, a, nb, block, smem, st);
#ifdef RTM_DEBUG
            case 16: return (c->opt_dbg & 32) ? launch_ex(c, acoustic3d_stream_kernel<16, false>, a, nb, block, smem, st)
                                              : launch_ex(c, acoustic3d_stream_kernel<16, true>, a, nb, block, smem, st);
#else
            case 16: return launch_ex(c, acoustic3d_stream_kernel<16, true>, a, nb, block, smem, st);
#endif
            default: return launch_ex(c, acoustic3d_stream_kernel<32, true>, a, nb, block, smem, st);
        }
    }
}

static int launch_flush(rtm_ctx *c, const float *hist, int ncur, const float *Z0, long long zstep, float *PZ, cudaStream_t st) {
    // two probed fields: the r field sits Nu floats behind the p field in every slot and plane group, i.e. it is nx more
    // rows of the same pitch
    Layout L = c->L;
    if (c->cfg.probe_fields == 2) { L.nx *= 2; L.Nu *= 2; }
    const long long tot = (long long)L.nx * L.ny * (L.upz / 4);
    const unsigned nb = (unsigned)((tot + 255) / 256);
    if (c->T <= 4) probe_flush_kernel<4><<<nb, 256, 0, st>>>(L, hist, ncur, Z0, zstep, c->zr, c->cfg.r, PZ);
    else if (c->T <= 8) probe_flush_kernel<8><<<nb, 256, 0, st>>>(L, hist, ncur, Z0, zstep, c->zr, c->cfg.r, PZ);
    else if (c->T <= 16) probe_flush_kernel<16><<<nb, 256, 0, st>>>(L, hist, ncur, Z0, zstep, c->zr, c->cfg.r, PZ);
    else probe_flush_kernel<32><<<nb, 256, 0, st>>>(L, hist, ncur, Z0, zstep, c->zr, c->cfg.r, PZ);
    c->launches++;
    return RTM_OK;
}

static int run_pass(rtm_ctx *c, int adjoint, const PassGeom &g, const float *d_inj_val, float *d_smp_out,
                    float *PZ, const float *Z, cudaStream_t st) {
    const rtm_config &cfg = c->cfg;
    const Layout &L = c->L;
    const int nt = cfg.nt, d = cfg.ndim, T = c->T;
    CU(cudaMemsetAsync(c->fields_base, 0, c->fields_bytes, st));
    CU(cudaMemsetAsync(PZ, 0, (size_t)c->rp * (size_t)L.Nu * 4, st));

    StepArgs a;
    memset(&a, 0, sizeof a);
    a.L = L;
    a.K2 = c->K2; a.epsh = c->epsh; a.delh = c->delh; a.cs = c->cs; a.sn = c->sn;
    a.cp = c->cp; a.sp = c->sp;
    for (int k = 0; k < 6; k++) a.F[k] = c->F[k];
    const bool tti3 = cfg.physics == 1 && d == 3;   // three kernels per step, no in-launch flush role: flush at the end of a time block
    a.dampx = c->dampx; a.dampy = c->dampy; a.dampz = c->dampz;
    a.k1x = c->k1x; a.k1y = c->k1y; a.k1z = c->k1z;
    a.adjoint = adjoint;
    a.PZ = PZ;
    a.r = cfg.r;
    a.two = cfg.probe_fields == 2;
    a.pNu = c->pNu;
    a.row_start = c->row_start;
    a.ent = c->ent;
    double inj_scale = adjoint ? (double)cfg.h * (double)cfg.h : std::pow((double)cfg.h, 2.0 - d);
    double smp_scale = adjoint ? std::pow((double)cfg.h, -(double)d) : 1.0;
    if (cfg.physics == 1) { if (adjoint) inj_scale *= 0.5; else smp_scale *= 0.5; }
    a.inj_scale = (float)inj_scale;
    a.smp_scale = (float)smp_scale;
    a.bx0 = g.bx0; a.bx1 = g.bx1; a.by0 = g.by0; a.by1 = g.by1; a.bz0 = g.bz0; a.bz1 = g.bz1;
    a.smp_idx = c->smp_idx;
    a.smp_w = c->smp_w;
    a.nsmp = g.nsmp;
    a.nc = g.nc;

    dim3 grid, block;
    size_t smem;
    step_grid(c, &grid, &block, &smem);
    const long long nblocks = (long long)grid.x * grid.y * grid.z;
    const long long bthreads = (long long)block.x * block.y * block.z;
    const int fl_vec = (c->rx && T <= 16) ? 4 : 2;   // floats per flush-role thread (flush_role4 in the 2D streaming kernel)
    const long long units = (long long)L.nx * L.ny * (L.upz / fl_vec) * (a.two ? 2 : 1);
    a.gx = grid.x; a.gy = grid.y;
    if (c->rx) a.gx = (unsigned)((L.Pz + 3) / 4);   // streaming kernel: quads per row
    a.zr = c->zr;
    a.fl_zstep = adjoint ? -(long long)c->zr : (long long)c->zr;
    const bool want_smp = d_smp_out != nullptr && g.nsmp > 0;
    const bool deferred = want_smp && (long long)g.nsmp <= nblocks * bthreads;
    const unsigned smp_blocks = (unsigned)((g.nsmp + 255) / 256);

    const int evs = (int)(c->ev_count[adjoint] % rtm_ctx::kEvRing);
    if (c->opt_time) CU(cudaEventRecord(c->ev[adjoint][evs][0], st));
    int cur = 0;
    const long long Np = (long long)L.Px * L.Py * L.Pzc;
#ifdef RTM_DEBUG
    a.dbg = c->opt_dbg;
    a.dbg_ts = c->dbg_ts;
#endif
    const int res_mode = ((c->opt_resident == 1 || c->opt_resident == 2) && c->res[0].nb > 0 && g.res_ok[0]) ? 0
                       : (c->opt_resident >= 2 && c->res[1].nb > 0 && g.res_ok[1]) ? 1 : -1;
    if (res_mode >= 0) {
        // Resident 2D kernel: one cooperative launch per time block (cut after a step whose field is wanted as a
        // snapshot), the fields stay in fld[0][0] / fld[0][2]; then the block's history is flushed into the planes.
        int step = 0;
        while (step < nt) {
            const int b = step / T, slot = step % T;
            int len = std::min(T - slot, nt - step);
            for (size_t q = 0; q < c->snap_steps.size() && c->snap_out; q++) {
                const int ss = adjoint ? nt - 1 - c->snap_steps[q] : c->snap_steps[q];
                if (ss >= step && ss < step + len) len = ss - step + 1;
            }
            const int n0 = adjoint ? nt - 1 - step : step;
            int rc_ = launch_resident(c, res_mode, a, adjoint, n0, len, 0, g, d_inj_val, d_smp_out,
                                      c->hist + ((size_t)(b & 1) * T + slot) * c->pNu, st);
            if (rc_) return rc_;
            step += len;
            const int nlast = adjoint ? nt - step : step - 1;
            if (step % T == 0 || step == nt) {
                const int nfirst = adjoint ? nt - 1 - b * T : b * T;
                launch_flush(c, c->hist + (size_t)(b & 1) * T * c->pNu, step - b * T, Z + (size_t)nfirst * c->zr, a.fl_zstep, PZ, st);
            }
            for (size_t q = 0; q < c->snap_steps.size(); q++)
                if (c->snap_steps[q] == nlast && c->snap_out) {
                    unpack_field_kernel<<<(unsigned)((Np + 255) / 256), 256, 0, st>>>(L, c->fld[0][0], c->snap_out + (long long)q * Np);
                    c->launches++;
                }
        }
        if (c->opt_time) { CU(cudaEventRecord(c->ev[adjoint][evs][1], st)); c->ev_count[adjoint]++; }
        CU(cudaGetLastError());
        c->snap_steps.clear();
        c->snap_out = nullptr;
        return RTM_OK;
    }
    for (int step = 0; step < nt; step++) {
        const int n = adjoint ? nt - 1 - step : step;
        const int nprev = adjoint ? n + 1 : n - 1;
        a.u0 = c->fld[0][cur]; a.n0 = c->fld[0][cur ^ 1]; a.d0 = c->fld[0][2];
        a.u1 = c->fld[1][cur]; a.n1 = c->fld[1][cur ^ 1]; a.d1 = c->fld[1][2];
        a.Zrow = Z + (size_t)n * c->zr;
        a.tmaps = c->tmaps;
        a.tm_u = cur;
        a.inj_val = d_inj_val + (size_t)n * g.ninj;
        a.smp_out = (deferred && step > 0) ? d_smp_out + (size_t)nprev * g.nsmp : nullptr;
        a.fl_blocks = 0;
        a.fl_q0 = a.fl_q1 = 0;
        if (T) {
            // time block b = step / T writes history slots [(b&1) T, (b&1) T + T); while it runs, the
            // previous block is flushed in len_b slices, one per step launch
            const int b = step / T, slot = step % T;
            a.hist = c->hist + ((size_t)(b & 1) * T + slot) * c->pNu;
            if (b >= 1 && !tti3) {
                const int len_b = std::min(T, nt - b * T);
                const int pb = b - 1;
                const int nfirst = adjoint ? nt - 1 - pb * T : pb * T;
                a.fl_hist = c->hist + (size_t)(pb & 1) * T * c->pNu;
                a.fl_Z0 = Z + (size_t)nfirst * c->zr;
                a.fl_n = T;
                // slices go to slots 1 .. len_b-1: their input (the previous block's last slot) is then at least two
                // launches old and the role needs no grid dependency; a block of one step flushes on slot 0, waiting
                const int nsl = len_b > 1 ? len_b - 1 : 1, sl = len_b > 1 ? slot - 1 : 0;
                a.fl_nowait = (len_b > 1 && c->opt_pdl) ? 1 : 0;
                if (sl >= 0) {
                    a.fl_q0 = units * sl / nsl;
                    a.fl_q1 = units * (sl + 1) / nsl;
                    a.fl_blocks = (int)((a.fl_q1 - a.fl_q0 + bthreads - 1) / bthreads);   // one unit per thread
                }
            }
        }
#ifdef RTM_DEBUG
        if ((c->opt_dbg & 3) == 1) a.fl_blocks = 0;
        a.dbg = c->opt_dbg;
        a.dbg_ts = c->dbg_ts;
#endif
        { int rc_ = launch_step(c, a, grid, block, smem, st); if (rc_) return rc_; }
        cur ^= 1;
        if (tti3 && T && (step + 1) % T == 0 && step != nt - 1) {
            const int fb = step / T;
            const int nfirst = adjoint ? nt - 1 - fb * T : fb * T;
            launch_flush(c, c->hist + (size_t)(fb & 1) * T * c->pNu, T, Z + (size_t)nfirst * c->zr, a.fl_zstep, PZ, st);
        }
        if (T && step == nt - 1) {   // the last time block has no following steps to hide behind
            const int fb = step / T, lenf = nt - fb * T;
            const int nfirst = adjoint ? nt - 1 - fb * T : fb * T;
            launch_flush(c, c->hist + (size_t)(fb & 1) * T * c->pNu, lenf, Z + (size_t)nfirst * c->zr, a.fl_zstep, PZ, st);
        }
        if (c->opt_time && step == nt - 1) { CU(cudaEventRecord(c->ev[adjoint][evs][1], st)); c->ev_count[adjoint]++; }
        if (want_smp && (!deferred || step == nt - 1)) {
            StepArgs s = a;   // sample the field just computed
            s.u0 = c->fld[0][cur]; s.u1 = c->fld[1][cur];
            s.smp_out = d_smp_out + (size_t)n * g.nsmp;
            sample_kernel<<<smp_blocks, 256, 0, st>>>(s);
            c->launches++;
        }
        for (size_t q = 0; q < c->snap_steps.size(); q++)
            if (c->snap_steps[q] == n && c->snap_out)
                for (int f = 0; f < c->nf; f++) {
                    unpack_field_kernel<<<(unsigned)((Np + 255) / 256), 256, 0, st>>>(
                        L, c->fld[f][cur], c->snap_out + ((long long)q * c->nf + f) * Np);
                    c->launches++;
                }
    }
    CU(cudaGetLastError());
    c->snap_steps.clear();
    c->snap_out = nullptr;
    return RTM_OK;
}

extern "C" int rtm_forward_probe(rtm_ctx *c, int nsrc, const float *h_src_xyz, const float *d_wav, int nrec,
                                 const float *h_rec_xyz, float *d_data_out, void *stream) {
    if (!c || nsrc < 1 || !h_src_xyz || !d_wav || nrec < 0 || (nrec > 0 && !h_rec_xyz)) return RTM_EINVAL;
    DeviceGuard guard(c->device);
    if (nsrc > c->cfg.max_pts || nrec > c->cfg.max_pts) return RTM_EINVAL;
    if (!c->have_model || !c->have_probes) return RTM_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    PassGeom g;
    int rc = build_geometry(c, 0, nsrc, h_src_xyz, nrec, h_rec_xyz, &g, st);
    if (rc) return rc;
    c->have_U = false;
    rc = run_pass(c, 0, g, d_wav, d_data_out, c->Uz, c->Zf, st);
    if (rc) return rc;
    c->have_U = true;
    c->have_V = false;
    return RTM_OK;
}

static int launch_image(rtm_ctx *c, float scale, int accumulate, float *d_image, cudaStream_t st) {
    const Layout &L = c->L;
    const long long tot = (long long)L.nx * L.ny * (L.upz / 4);
    image_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(L, c->Uz, c->Vz, c->rp, scale, accumulate, d_image);
    c->launches++;
    CU(cudaGetLastError());
    return RTM_OK;
}

extern "C" int rtm_adjoint_image(rtm_ctx *c, int nrec, const float *h_rec_xyz, const float *d_data_in, int nsrc,
                                 const float *h_src_xyz, float *d_qadj_out, float scale, int accumulate,
                                 float *d_image, void *stream) {
    if (!c || nrec < 1 || !h_rec_xyz || !d_data_in || nsrc < 0 || (nsrc > 0 && !h_src_xyz)) return RTM_EINVAL;
    DeviceGuard guard(c->device);
    if (nsrc > c->cfg.max_pts || nrec > c->cfg.max_pts) return RTM_EINVAL;
    if (!c->have_model || !c->have_probes) return RTM_ESTATE;
    if (d_image && !c->have_U) return RTM_ESTATE;   // adjoint before forward
    cudaStream_t st = (cudaStream_t)stream;
    PassGeom g;
    int rc = build_geometry(c, 1, nrec, h_rec_xyz, nsrc, h_src_xyz, &g, st);
    if (rc) return rc;
    c->have_V = false;
    rc = run_pass(c, 1, g, d_data_in, d_qadj_out, c->Vz, c->Za, st);
    if (rc) return rc;
    c->have_V = true;
    if (d_image) return launch_image(c, scale, accumulate, d_image, st);
    return RTM_OK;
}

extern "C" int rtm_image(rtm_ctx *c, float scale, int accumulate, float *d_image, void *stream) {
    if (!c || !d_image) return RTM_EINVAL;
    DeviceGuard guard(c->device);
    if (!c->have_U || !c->have_V) return RTM_ESTATE;
    return launch_image(c, scale, accumulate, d_image, (cudaStream_t)stream);
}

extern "C" int rtm_offset_gather(rtm_ctx *c, int nh, const int *h_offsets, float scale, float *d_gather, void *stream) {
    if (!c || nh < 1 || nh > 4096 || !h_offsets || !d_gather) return RTM_EINVAL;
    DeviceGuard guard(c->device);
    if (!c->have_U || !c->have_V) return RTM_ESTATE;
    for (int i = 0; i < nh; i++)
        if (std::abs(h_offsets[i]) >= c->cfg.n[0]) return RTM_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    if (c->offs_pending) { CU(cudaEventSynchronize(c->offs_done)); c->offs_pending = false; }
    memcpy(c->h_offs, h_offsets, (size_t)nh * 4);
    CU(cudaMemcpyAsync(c->offs, c->h_offs, (size_t)nh * 4, cudaMemcpyHostToDevice, st));
    CU(cudaEventRecord(c->offs_done, st));
    c->offs_pending = true;
    const Layout &L = c->L;
    bool run = nh >= 8 && nh <= GT_HP;   // a run of consecutive offsets takes the register-tiled kernel
    for (int i = 1; i < nh && run; i++) run = h_offsets[i] == h_offsets[i - 1] + 1;
    if (run) {
        const dim3 grid((unsigned)(((long long)L.ny * L.upz) / 32), (unsigned)((L.nx + GT_X - 1) / GT_X), 1);
        if (nh > 16) CU(optin_max_smem((const void *)gather_tiled_kernel<GT_HP, false>, c->device));   // 81 KB of staging: 4 probes in flight
        if (nh <= 16) gather_tiled_kernel<16, false><<<grid, gt_threads(16), gt_smem(16), st>>>(L, c->Uz, c->Vz, c->rp, nh, h_offsets[0], nullptr, 0, scale, d_gather);
        else gather_tiled_kernel<GT_HP, false><<<grid, gt_threads(GT_HP), gt_smem(GT_HP), st>>>(L, c->Uz, c->Vz, c->rp, nh, h_offsets[0], nullptr, 0, scale, d_gather);
    } else {
        const long long tot = (long long)L.nx * L.ny * (L.upz / 4);
        gather_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(L, c->Uz, c->Vz, c->rp, nh, c->offs, scale, d_gather);
    }
    c->launches++;
    CU(cudaGetLastError());
    return RTM_OK;
}

extern "C" int rtm_offset_gather_xy(rtm_ctx *c, int nh, const int *h_offsets_xy, float scale, float *d_gather, void *stream) {
    if (!c || nh < 1 || nh > 4096 || !h_offsets_xy || !d_gather || c->cfg.ndim != 3) return RTM_EINVAL;
    DeviceGuard guard(c->device);
    if (!c->have_U || !c->have_V) return RTM_ESTATE;
    for (int i = 0; i < nh; i++)
        if (std::abs(h_offsets_xy[2 * i]) >= c->cfg.n[0] || std::abs(h_offsets_xy[2 * i + 1]) >= c->cfg.n[1]) return RTM_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    const Layout &L = c->L;
    if (c->offs_pending) { CU(cudaEventSynchronize(c->offs_done)); c->offs_pending = false; }
    // runs of consecutive hx at one hy (8..GT_HP long) take the register-tiled kernel -- one launch for all runs of up
    // to 16 offsets, one for the longer ones -- the rest go to the generic kernel as (ih, hx, hy) triples
    int nl = 0, nrun[2] = {0, 0};
    int *trip = c->h_offs, *run[2] = {c->h_offs + 3 * 4096, c->h_offs + 4 * 4096};
    for (int i = 0; i < nh;) {
        int j = i + 1;
        while (j < nh && j - i < GT_HP && h_offsets_xy[2 * j + 1] == h_offsets_xy[2 * i + 1] &&
               h_offsets_xy[2 * j] == h_offsets_xy[2 * (j - 1)] + 1)
            j++;
        if (j - i >= 8) {
            const int cls = j - i <= 16 ? 0 : 1;
            int *rec = run[cls] + 4 * nrun[cls]++;
            rec[0] = h_offsets_xy[2 * i]; rec[1] = h_offsets_xy[2 * i + 1]; rec[2] = j - i; rec[3] = i;
        } else {
            for (int m = i; m < j; m++) {
                trip[3 * nl] = m;
                trip[3 * nl + 1] = h_offsets_xy[2 * m];
                trip[3 * nl + 2] = h_offsets_xy[2 * m + 1];
                nl++;
            }
        }
        i = j;
    }
    CU(cudaMemcpyAsync(c->offs, c->h_offs, (size_t)5 * 4096 * 4, cudaMemcpyHostToDevice, st));
    CU(cudaEventRecord(c->offs_done, st));
    c->offs_pending = true;
    for (int cls = 0; cls < 2; cls++) {
        if (!nrun[cls]) continue;
        const long long nblk = (long long)L.ny * (L.upz / 32) * ((L.nx + GT_X - 1) / GT_X) * nrun[cls];
        if (nblk >= (1LL << 31)) return RTM_EINVAL;
        const int4 *d_runs = (const int4 *)(c->offs + (3 + cls) * 4096);
        if (cls == 0)
            gather_tiled_kernel<16, true><<<(unsigned)nblk, gt_threads(16), gt_smem(16), st>>>(L, c->Uz, c->Vz, c->rp, 0, 0, d_runs, nrun[cls], scale, d_gather);
        else {
            CU(optin_max_smem((const void *)gather_tiled_kernel<GT_HP, true>, c->device));
            gather_tiled_kernel<GT_HP, true><<<(unsigned)nblk, gt_threads(GT_HP), gt_smem(GT_HP), st>>>(L, c->Uz, c->Vz, c->rp, 0, 0, d_runs, nrun[cls], scale, d_gather);
        }
        c->launches++;
    }
    if (nl) {
        const long long tot = (long long)L.nx * L.ny * (L.upz / 4);
        gather_xy_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(L, c->Uz, c->Vz, c->rp, nl, c->offs, scale, d_gather);
        c->launches++;
    }
    CU(cudaGetLastError());
    return RTM_OK;
}

extern "C" size_t rtm_shot_staging_bytes(const rtm_config *cfg, int nsrc, int nrec, int nh) {
    if (!valid_cfg(cfg) || nsrc < 1 || nrec < 1 || nh < 0) return 0;
    Layout L;
    make_layout(cfg, &L);
    const size_t N = (size_t)L.nx * L.ny * L.nz, nt = (size_t)cfg->nt;
    size_t b = 0;
    b += (size_t)rup((long long)(nt * nsrc * 4), 256);
    b += 2 * (size_t)rup((long long)(nt * nrec * 4), 256);
    b += (size_t)rup((long long)(N * 4), 256);
    b += (size_t)rup((long long)((size_t)nh * N * 4), 256);
    return b + 256;
}

extern "C" int rtm_shot_host(rtm_ctx *c, int nsrc, const float *h_src_xyz, const float *h_wav, int nrec,
                             const float *h_rec_xyz, const float *h_data_in, float *h_data_out, float scale,
                             float *h_image, int nh, const int *h_offsets, float *h_gather, void *d_staging,
                             size_t staging_bytes, void *stream) {
    if (!c || !h_wav || !h_data_in || !d_staging) return RTM_EINVAL;
    DeviceGuard guard(c->device);
    // everything a later stage would reject is rejected before any work is enqueued
    if (nsrc < 1 || nrec < 1 || !h_src_xyz || !h_rec_xyz || nsrc > c->cfg.max_pts || nrec > c->cfg.max_pts) return RTM_EINVAL;
    if (nh < 0 || nh > 4096 || (nh > 0 && h_gather && !h_offsets)) return RTM_EINVAL;
    for (int i = 0; i < nh && h_gather; i++)
        if (std::abs(h_offsets[i]) >= c->cfg.n[0]) return RTM_EINVAL;
    if (!c->have_model || !c->have_probes) return RTM_ESTATE;
    {
        Corner co[8];
        for (int s = 0; s < nsrc; s++) if (corners_of(c->cfg, c->L, h_src_xyz + (size_t)s * c->cfg.ndim, co) < 0) return RTM_EINVAL;
        for (int s = 0; s < nrec; s++) if (corners_of(c->cfg, c->L, h_rec_xyz + (size_t)s * c->cfg.ndim, co) < 0) return RTM_EINVAL;
    }
    size_t need = rtm_shot_staging_bytes(&c->cfg, nsrc, nrec, nh);
    if (need == 0 || ((uintptr_t)d_staging & 255)) return RTM_EINVAL;
    if (staging_bytes < need) return RTM_ENOMEM;
    cudaStream_t st = (cudaStream_t)stream;
    const Layout &L = c->L;
    const size_t N = (size_t)L.nx * L.ny * L.nz, nt = (size_t)c->cfg.nt;
    char *p = (char *)d_staging;
    float *d_wav = (float *)p;  p += rup((long long)(nt * nsrc * 4), 256);
    float *d_din = (float *)p;  p += rup((long long)(nt * nrec * 4), 256);
    float *d_dout = (float *)p; p += rup((long long)(nt * nrec * 4), 256);
    float *d_img = (float *)p;  p += rup((long long)(N * 4), 256);
    float *d_gat = (float *)p;
    CU(cudaMemcpyAsync(d_wav, h_wav, nt * nsrc * 4, cudaMemcpyHostToDevice, st));
    CU(cudaMemcpyAsync(d_din, h_data_in, nt * nrec * 4, cudaMemcpyHostToDevice, st));
    int rc = rtm_forward_probe(c, nsrc, h_src_xyz, d_wav, nrec, h_rec_xyz, h_data_out ? d_dout : nullptr, stream);
    if (rc) return rc;
    if (h_data_out) CU(cudaMemcpyAsync(h_data_out, d_dout, nt * nrec * 4, cudaMemcpyDeviceToHost, st));
    rc = rtm_adjoint_image(c, nrec, h_rec_xyz, d_din, nsrc, h_src_xyz, nullptr, scale, 0, h_image ? d_img : nullptr, stream);
    if (rc) return rc;
    if (h_image) CU(cudaMemcpyAsync(h_image, d_img, N * 4, cudaMemcpyDeviceToHost, st));
    if (nh > 0 && h_gather) {
        rc = rtm_offset_gather(c, nh, h_offsets, scale, d_gat, stream);
        if (rc) return rc;
        CU(cudaMemcpyAsync(h_gather, d_gat, (size_t)nh * N * 4, cudaMemcpyDeviceToHost, st));
    }
    return RTM_OK;
}

// ---- test hooks ----------------------------------------------------------------------------------
extern "C" int rtm_export_probes(rtm_ctx *c, int which, float *d_out, void *stream) {
    if (!c || !d_out || (which != 0 && which != 1)) return RTM_EINVAL;
    DeviceGuard guard(c->device);
    if (which == 0 ? !c->have_U : !c->have_V) return RTM_ESTATE;
    const Layout &L = c->L;
    const long long tot = (long long)L.nx * L.ny * L.nz * c->rp;
    unpack_probes_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, (cudaStream_t)stream>>>(L, c->rp, c->cfg.probe_fields == 2, which ? c->Vz : c->Uz, d_out);
    c->launches++;
    CU(cudaGetLastError());
    return RTM_OK;
}

extern "C" int rtm_set_snapshots(rtm_ctx *c, int nsnap, const int *h_steps, float *d_out) {
    if (!c || nsnap < 0 || (nsnap > 0 && (!h_steps || !d_out))) return RTM_EINVAL;
    c->snap_steps.assign(h_steps, h_steps + nsnap);
    c->snap_out = nsnap ? d_out : nullptr;
    return RTM_OK;
}

extern "C" int rtm_export_coeff(rtm_ctx *c, int which, float *d_out, void *stream) {
    if (!c || !d_out || which < 0 || which > 6) return RTM_EINVAL;
    DeviceGuard guard(c->device);
    if (!c->have_model) return RTM_ESTATE;
    const float *src[7] = {c->K2, c->epsh, c->delh, c->cs, c->sn, c->cp, c->sp};
    if (!src[which]) return RTM_EINVAL;
    const long long Np = (long long)c->L.Px * c->L.Py * c->L.Pzc;
    unpack_field_kernel<<<(unsigned)((Np + 255) / 256), 256, 0, (cudaStream_t)stream>>>(c->L, src[which], d_out);
    c->launches++;
    CU(cudaGetLastError());
    return RTM_OK;
}

extern "C" float rtm_pass_ms_mean(rtm_ctx *c, int which, int count) {
    if (!c || (which != 0 && which != 1) || count < 1 || count > rtm_ctx::kEvRing || c->ev_count[which] < count) return -1.0f;
    DeviceGuard guard(c->device);
    double sum = 0.0;
    for (int i = 1; i <= count; i++) {
        const int s = (int)((c->ev_count[which] - i) % rtm_ctx::kEvRing);
        if (cudaEventSynchronize(c->ev[which][s][1]) != cudaSuccess) return -1.0f;
        float ms = -1.0f;
        if (cudaEventElapsedTime(&ms, c->ev[which][s][0], c->ev[which][s][1]) != cudaSuccess) return -1.0f;
        sum += ms;
    }
    return (float)(sum / count);
}
extern "C" float rtm_last_pass_ms(rtm_ctx *c, int which) { return rtm_pass_ms_mean(c, which, 1); }

#ifdef RTM_DEBUG
// timing experiments: copy the per-block phase stamps of the last launch (dbg & 16) to the host; synchronises
extern "C" int rtm_debug_stamps(rtm_ctx *c, unsigned long long *h_out, int nblocks) {
    if (!c || !h_out || nblocks < 1 || nblocks > 1024) return RTM_EINVAL;
    DeviceGuard guard(c->device);
    CU(cudaDeviceSynchronize());
    CU(cudaMemcpy(h_out, c->dbg_ts, (size_t)nblocks * 8 * 8, cudaMemcpyDeviceToHost));
    return RTM_OK;
}
#endif

extern "C" long long rtm_launch_count(const rtm_ctx *c) { return c ? c->launches : 0; }

extern "C" int rtm_set_option(rtm_ctx *c, const char *name, int value) {
    if (!c || !name) return RTM_EINVAL;
    if (!strcmp(name, "time_steps")) { c->opt_time = value; return RTM_OK; }
    if (!strcmp(name, "pdl")) { c->opt_pdl = value; return RTM_OK; }
#ifdef RTM_DEBUG
    if (!strcmp(name, "dbg")) { c->opt_dbg = value; return RTM_OK; }   // timing experiments only: 1 = no flush role, 2 = no stencil
#endif
    if (!strcmp(name, "resident")) {   // 2D acoustic, T > 1: wavefield resident in shared memory for a whole time block
        if (value < 0 || value > 3) return RTM_EINVAL;
        c->opt_resident = value;
        return RTM_OK;
    }
    if (!strcmp(name, "tti_tile")) {   // 2D TTI, time blocks of 9..16 steps: rows per tile of the step kernel, 16 or 32
        if (c->cfg.ndim != 2 || c->cfg.physics != 1 || (value != 16 && value != 32)) return RTM_EINVAL;
        if (value == 32 && tm_of(c->T) != 16) return RTM_EINVAL;   // the 32-row instance exists for T in 9..16 only
        c->tti_tx = value;
        return RTM_OK;
    }
    if (!strcmp(name, "rx")) {   // rows per thread of the 2D streaming kernel (2|4|8|16); 0 = automatic
        if (!c->rx) return RTM_EINVAL;
        if (value != 0 && value != 2 && value != 4 && value != 8 && value != 16) return RTM_EINVAL;   // the kernel's instances
        DeviceGuard guard(c->device);
        c->rx = value > 0 ? value : pick_rx(c);
        return RTM_OK;
    }
    return RTM_EINVAL;
}

// ---- the entry point that allocates nothing (rtm.h: rtm_offset_gather_static) --------------------------------------
// The operands of gather_kernel (image.cuh) -- U and V in rows of upz floats, the offsets table -- are workspace memory in
// a context; here they live in a file-scope device array, so the call needs no context and no allocation.  In host code
// the NAME g_static_scratch is only a stand-in for the symbol (not a device address): the address comes from
// cudaGetSymbolAddress, once per device, with that device current, and is what the kernels are given.
static __device__ __align__(256) float g_static_scratch[RTM_STATIC_SCRATCH_BYTES / 4];
static std::mutex g_static_mu;
static float *g_static_ptr[64];   // device address of g_static_scratch, per device ordinal

struct StaticOffsets { int h[RTM_STATIC_MAX_OFFSETS]; };

// [planes][nx][nz] of U and of V -> rows of upz floats in the scratch (pad columns are WRITTEN as zeros: the array keeps
// the previous call's contents); the first nh threads also store the offsets table, which arrives as a kernel argument
__global__ void __launch_bounds__(256) static_pack_kernel(int nz, int upz, long long rows, const float *__restrict__ U,
                                                          const float *__restrict__ V, float *__restrict__ sU,
                                                          float *__restrict__ sV, int *__restrict__ sOffs, int nh,
                                                          const __grid_constant__ StaticOffsets offs) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t < nh) sOffs[t] = offs.h[t];
    if (t >= rows * upz) return;
    const int iz = (int)(t % upz);
    const long long row = t / upz;
    const bool in = iz < nz;
    sU[t] = in ? U[row * nz + iz] : 0.0f;
    sV[t] = in ? V[row * nz + iz] : 0.0f;
}

static int static_scratch_address(float **out) {
    int dev = -1;
    CU(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) return RTM_EINVAL;
    std::lock_guard<std::mutex> lk(g_static_mu);
    if (!g_static_ptr[dev]) {
        void *p = nullptr;
        CU(cudaGetSymbolAddress(&p, g_static_scratch));
        g_static_ptr[dev] = (float *)p;
    }
    *out = g_static_ptr[dev];
    return RTM_OK;
}

extern "C" int rtm_offset_gather_static(int nx, int nz, int r, const float *d_U, const float *d_V, int nh, const int *h_offsets,
                                        float scale, float *d_gather, void *stream) {
    if (nx < 1 || nz < 1 || r < 1 || nh < 1 || !d_U || !d_V || !h_offsets || !d_gather) return RTM_EINVAL;
    if (nh > RTM_STATIC_MAX_OFFSETS) return RTM_ELIMIT;
    const long long cap = (long long)(RTM_STATIC_SCRATCH_BYTES / 4) - 64;   // floats after the offsets table (256 B)
    const long long upz = rup(nz, 4);
    if (upz > cap || nx > cap / upz || r > cap / (2 * upz * nx)) return RTM_ELIMIT;
    StaticOffsets offs;
    for (int i = 0; i < nh; i++) {
        if (std::abs((long long)h_offsets[i]) >= nx) return RTM_EINVAL;
        offs.h[i] = h_offsets[i];
    }
    for (int i = nh; i < RTM_STATIC_MAX_OFFSETS; i++) offs.h[i] = 0;
    float *scratch = nullptr;
    int rc = static_scratch_address(&scratch);
    if (rc) return rc;
    int *sOffs = reinterpret_cast<int *>(scratch);
    float *sU = scratch + 64, *sV = sU + (long long)r * nx * upz;
    Layout L{};
    L.nd = 2; L.nx = nx; L.ny = 1; L.nz = nz;
    L.upz = (int)upz;
    L.Nu = (long long)nx * upz;
    cudaStream_t st = (cudaStream_t)stream;
    const long long rows = (long long)r * nx, tot = std::max(rows * upz, (long long)nh);
    static_pack_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>((int)nz, (int)upz, rows, d_U, d_V, sU, sV, sOffs, nh, offs);
    const long long quads = (long long)nx * (upz / 4);
    gather_kernel<<<(unsigned)((quads + 255) / 256), 256, 0, st>>>(L, sU, sV, r, nh, sOffs, scale, d_gather);
    CU(cudaGetLastError());
    return RTM_OK;
}

extern "C" const char *rtm_strerror(int code) {
    switch (code) {
        case RTM_OK: return "ok";
        case RTM_EINVAL: return "invalid argument";
        case RTM_ENOMEM: return "workspace too small";
        case RTM_ECUDA: return "CUDA error";
        case RTM_ESTATE: return "call out of order";
        case RTM_ELIMIT: return "size beyond the static scratch (RTM_STATIC_SCRATCH_BYTES / RTM_STATIC_MAX_OFFSETS in rtm.h)";
        default: return "unknown error";
    }
}
extern "C" const char *rtm_last_cuda_error(void) { return g_cuda_err; }
