/*
 * rtm.h -- C ABI of the B200 (sm_100a) RTM-with-randomized-trace-imaging hot path.
 *
 * Method: Louboutin & Herrmann, "Enabling wave-based inversion on GPUs with randomized trace
 * estimation" (arXiv 2201.06914); citations are PAPER.md:Lnn (+ section / equation).
 * The paper fixes the estimator (Eq. 1), the imaging conditions (Eq. 2-4) and the
 * O(N r) memory claim (L47, Table 1).  It gives no discretisation; DESIGN.md "Readings"
 * fixes the FD scheme, boundary, source/receiver handling.
 *
 * Conventions
 *   - plain C, no exceptions cross the ABI; every call returns 0 or a negative RTM_E* code.
 *   - pointer prefix d_ = device memory, h_ = host memory.  The caller owns every buffer,
 *     including the workspace; the library allocates and frees no device memory.
 *   - all device work is enqueued on the `cuda_stream` argument (a cudaStream_t passed as void*);
 *     no call synchronises the device.  Host tables (geometry, offsets) are built synchronously on the host
 *     in pinned staging buffers of the context and uploaded with cudaMemcpyAsync on the same stream; a call
 *     that needs a staging buffer whose previous upload (the previous call of the same kind) has not been
 *     consumed yet waits on the host for that one copy (cudaEventSynchronize), never for kernels of its own.
 *   - every call runs on the device that owns the workspace (taken from the pointer at rtm_create); the calling
 *     thread's current device is restored on return.
 *   - grids: physical grid n = (nx,[ny],nz), z contiguous (C order [x][z] / [x][y][z]); absorbing
 *     layer of nb points on every side; padded grid P = n + 2 nb, Np = prod P, N = prod n.
 *     "canonical [Np]" / "[N]" arrays are dense C-order arrays without halo or pitch.
 *   - fp32 storage and arithmetic on the device.
 */
#ifndef RTM_H
#define RTM_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

#define RTM_OK 0
#define RTM_EINVAL (-1) /* bad shape / NULL / position outside the physical grid / bad offset   */
#define RTM_ENOMEM (-2) /* workspace too small                                                  */
#define RTM_ECUDA (-3)  /* a CUDA call failed; text via rtm_last_cuda_error()                   */
#define RTM_ESTATE (-4) /* call order: adjoint before forward, gather before adjoint, no model  */

typedef struct rtm_ctx rtm_ctx; /* opaque, host-side */

typedef struct {
    int ndim;       /* 2 | 3 */
    int n[3];       /* physical points: 2D (nx, nz, -) ; 3D (nx, ny, nz); z contiguous            */
    float h;        /* grid spacing [m], same on every axis                                       */
    int nb;         /* absorbing-layer points on every side, 0..1024 (any value: the internal z axis is
                       shifted so that the physical grid stays float4-aligned)                      */
    int physics;    /* 0 isotropic acoustic ; 1 pseudo-acoustic TTI (2D: tilt; 3D: tilt + azimuth,
                       use rtm_coeffs_host3 / rtm_set_model3)                                    */
    int nt;         /* time steps                                                                 */
    double dt;      /* time step [s] (used by rtm_coeffs_host only, which rejects dt <= 0 / non-finite) */
    int r;          /* number of probing vectors, 1..256 (Eq. 1)                    */
    int max_pts;    /* upper bound on nsrc and nrec of any later call (sizes geometry tables)     */
    int probe_block;/* T_b: 0|1 = probe fused into every time step (8 r bytes/point/step of Uz traffic);
                       2..16 (2..32 for acoustic physics with r <= 128) = time-blocked probing: each step stores its field into a T_b-slot history
                       ring and every T_b steps one flush applies T_b rows of Z (traffic / T_b).
                       Same sums, same order per (k,x); costs 2 T_b N floats of workspace (the ring is
                       double-buffered: one half is filled while the other is flushed).             */
    int probe_fields;/* 0|1: one probed field per pass (TTI: 1/2 (p + r), reading C10).
                       2 (physics 1 only, 2D and 3D; any probe_block): the exact TTI gradient's four compressed arrays
                       (Eq. 2-3, on the coupled (p, r) system of L77; reading C29): every pass probes
                       p and r apart with the same Z, Uz = (Pz, Rz), Vz = (Wpz, Wrz), 2r planes each; the image and
                       the gathers sum over the 2r planes, scale = 1/r; rtm_export_probes returns [2r][N] (p planes, then
                       r planes).  Doubles the probe planes and the history ring.                            */
} rtm_config;

/* Bytes of device workspace rtm_create needs for this config; 0 if the config is invalid.
 * Holds: wavefields (u ping-pong + increment; x2 for TTI), coefficient arrays, damping tables,
 * the compressed wavefields Uz and Vz (2 r N floats: the O(N r) storage of PAPER.md:L47 / Table 1),
 * probe matrices (2 nt r), geometry tables.                                                       */
size_t rtm_workspace_bytes(const rtm_config *cfg);

/* Create a context over a caller-owned device workspace (256-byte aligned, >= rtm_workspace_bytes).
 * Errors: RTM_EINVAL (bad config / NULL / misaligned), RTM_ENOMEM (bytes too small).              */
int rtm_create(const rtm_config *cfg, void *d_workspace, size_t bytes, rtm_ctx **out);
void rtm_destroy(rtm_ctx *ctx);

/* Host helper: coefficient arrays of the scheme (1/c^2)(u_tt + 2 sigma u_t) - Lap u = q from the
 * earth model (O1).  fp64 arithmetic, one rounding to fp32.  Inputs are canonical [N]
 * host arrays (eps/delta/theta may be NULL for physics 0); outputs canonical [Np] host arrays
 * (TTI outputs may be NULL for physics 0) and h_damp1d = per-axis tables sigma_a*dt concatenated
 * over the axes (Px [+Py] +Pz floats).                                                           */
int rtm_coeffs_host(const rtm_config *cfg, const float *h_vp, const float *h_eps, const float *h_delta,
                    const float *h_theta, float *h_K2, float *h_epsh, float *h_delh, float *h_cos,
                    float *h_sin, float *h_damp1d);

/* 3D TTI ("TTI", L81 "generalize to 3D"; reading C30): the symmetry axis is
 * n = (sin th cos ph, sin th sin ph, cos th) with tilt th (h_theta) from the z axis and azimuth ph (h_phi) from the x
 * axis, both canonical [N] host arrays in radians.  As rtm_coeffs_host, plus h_cosp / h_sinp = cos / sin of ph [Np].
 * Errors: RTM_EINVAL (physics != 1 or ndim != 3, NULL, bad dt).                                                       */
int rtm_coeffs_host3(const rtm_config *cfg, const float *h_vp, const float *h_eps, const float *h_delta,
                     const float *h_theta, const float *h_phi, float *h_K2, float *h_epsh, float *h_delh,
                     float *h_cos, float *h_sin, float *h_cosp, float *h_sinp, float *h_damp1d);

/* Load the coefficient arrays (canonical [Np] DEVICE arrays; TTI ones NULL for physics 0) and the
 * per-axis damping tables (HOST) into the workspace's internal (haloed, pitched) layout.         */
int rtm_set_model(rtm_ctx *ctx, const float *d_K2, const float *d_epsh, const float *d_delh,
                  const float *d_cos, const float *d_sin, const float *h_damp1d, void *cuda_stream);

/* The same for a 3D TTI context (d_cosp, d_sinp: cos / sin of the azimuth, canonical [Np] DEVICE arrays).  A 3D TTI
 * context rejects rtm_set_model (RTM_EINVAL); every other context rejects this call.                                  */
int rtm_set_model3(rtm_ctx *ctx, const float *d_K2, const float *d_epsh, const float *d_delh, const float *d_cos,
                   const float *d_sin, const float *d_cosp, const float *d_sinp, const float *h_damp1d, void *cuda_stream);

/* Probing matrices Z (reading C1/C2: E[z z^T] = I, drawn by the caller), device
 * arrays [nt][r]; row n probes the field computed by step n (reading C6).  Zf is used by the
 * forward pass, Za by the adjoint pass (may alias; separate so that Eq. 3's u_tt can be had by
 * differencing Z, reading C4).  Copied into the workspace.                                        */
int rtm_set_probes(rtm_ctx *ctx, const float *d_Zf, const float *d_Za, void *cuda_stream);

/* Host helper for Eq. 2-3's gradient-type imaging condition  sum_t u_tt(t) v(t)  (reading C4):
 * with w[n] the field computed by step n,  sum_n z[n] (w[n] - 2 w[n-1] + w[n-2]) / dt^2  =  sum_n Zdd[n] w[n],
 *   Zdd[n][k] = (Z[n][k] - 2 Z[n+1][k] + Z[n+2][k]) / dt^2,   Z[nt] = Z[nt+1] = 0,
 * so probing u_tt costs nothing: pass Zdd as d_Zf and Z as d_Za to rtm_set_probes.  fp64 arithmetic, one rounding
 * to fp32.  h_Z, h_Zdd: HOST arrays [nt][r] (may not alias).  Errors: RTM_EINVAL.                      */
int rtm_probes_dtt_host(int nt, int r, double dt, const float *h_Z, float *h_Zdd);

/* Range-finder probes ("[Q, ~] = qr(A Z) where Z is a Rademacher random matrix"; refs [21, 26, 27];
 * DESIGN.md reading C3): A = D D^T, the nt x nt temporal covariance of the shot record h_D [nt][nrec] the adjoint
 * pass back-propagates (never formed); h_Q [nt][r] = orthonormal factor of the thin QR of D (D^T Z), diag(R) > 0.
 * Q^T Q = I_r: pass h_Q to rtm_set_probes (upload it first) and use scale = 1.0f, not 1/r (u^T Q Q^T v is a
 * projection).  Host pointers, fp64 arithmetic, one rounding to fp32.  Errors: RTM_EINVAL (r > nt, NULL, h_Q == h_Z,
 * or D (D^T Z) numerically rank-deficient, e.g. r > rank D).                                                    */
int rtm_probes_qr_host(int nt, int nrec, int r, const float *h_D, const float *h_Z, float *h_Q);

/* Forward pass with fused probing (Eq. 3: u_bar = Z^T u accumulated on the fly).
 * Zeroes the wavefields and Uz, runs n = 0..nt-1:  time step with fused damping; inject
 * K2 h^(2-d) w wav[n][s] at the 2^d corners of each source; record d[n][j] = sum_c w u[corner];
 * Uz[k][x] += Zf[n][k] u[x] on the physical grid.  Leaves Uz in the context.
 *   h_src_xyz [nsrc][ndim], h_rec_xyz [nrec][ndim]: metres from the physical origin (HOST);
 *   d_wav [nt][nsrc] (DEVICE); d_data_out [nt][nrec] (DEVICE) or NULL.
 * Errors: RTM_EINVAL (NULL, counts > max_pts, a position outside [0,(n_a-1)h]), RTM_ESTATE.       */
int rtm_forward_probe(rtm_ctx *ctx, int nsrc, const float *h_src_xyz, const float *d_wav, int nrec,
                      const float *h_rec_xyz, float *d_data_out, void *cuda_stream);

/* Adjoint pass with fused probing, then the image (Eq. 2-3).
 * Zeroes the wavefields and Vz, runs n = nt-1..0: time step; inject K2 h^2 w din[n][j] at the
 * receivers; optionally record qadj[n][s] = h^-d sum_c w v[corner] at the sources (exact transpose
 * of the forward map wav -> data); Vz[k][x] += Za[n][k] v[x].  Then
 *   image[x] (+)= scale * sum_k Uz[k][x] Vz[k][x]            (pass scale = 1/r for Eq. 3).
 *   d_data_in [nt][nrec]; d_qadj_out [nt][nsrc] or NULL; d_image canonical [N] or NULL
 *   (NULL: only Vz is formed); accumulate != 0 adds into d_image (stacking shots, L54/L77).       */
int rtm_adjoint_image(rtm_ctx *ctx, int nrec, const float *h_rec_xyz, const float *d_data_in, int nsrc,
                      const float *h_src_xyz, float *d_qadj_out, float scale, int accumulate,
                      float *d_image, void *cuda_stream);

/* The image alone, from the compressed wavefields the last forward and adjoint passes left in the context
 * (Eq. 3):  image[x] (+)= scale * sum_k Uz[k][x] Vz[k][x].  Same kernel and same bits as the image
 * rtm_adjoint_image writes; lets a caller re-image with another scale, or stack, without a new pass.
 *   d_image canonical [N] (DEVICE).  Errors: RTM_EINVAL (NULL), RTM_ESTATE (no Uz/Vz yet).               */
int rtm_image(rtm_ctx *ctx, float scale, int accumulate, float *d_image, void *cuda_stream);

/* Horizontal subsurface-offset volumes (Eq. 4; reading C11):
 *   gather[ih][x] = scale * sum_k Uz[k][x + h e_x] Vz[k][x - h e_x],  h = h_offsets[ih] grid points
 *   along x, zero where x+h or x-h leaves [0,nx).  gather[h=0] == image (L52).
 *   d_gather [nh][N].  Errors: RTM_EINVAL (nh < 1, |h| >= nx), RTM_ESTATE (no Uz/Vz yet).         */
int rtm_offset_gather(rtm_ctx *ctx, int nh, const int *h_offsets, float scale, float *d_gather,
                      void *cuda_stream);

/* Eq. 4 with VECTOR horizontal offsets on 3D grids ("h is a vector of horizontal offsets",
 * L81 "generalize to 3D", reading C28):
 *   gather[ih][x] = scale * sum_k Uz[k][x + hx e_x + hy e_y] Vz[k][x - hx e_x - hy e_y],
 *   (hx, hy) = h_offsets_xy[2 ih], h_offsets_xy[2 ih + 1] in grid points (host, [nh][2]); zero where either shifted
 *   point leaves [0,nx) x [0,ny).  (hx, 0) equals rtm_offset_gather bit for bit, (0, 0) the image.
 *   d_gather [nh][N] device, caller-owned.  Runs of >= 8 consecutive hx at one hy are served by the register-tiled
 *   kernel.  Errors: RTM_EINVAL (ndim != 3, nh < 1 or > 4096, |hx| >= nx, |hy| >= ny), RTM_ESTATE (no Uz/Vz yet).  */
int rtm_offset_gather_xy(rtm_ctx *ctx, int nh, const int *h_offsets_xy, float scale, float *d_gather,
                         void *cuda_stream);

/* One whole shot from HOST buffers (the end-to-end call): uploads wav and data_in, runs
 * rtm_forward_probe, rtm_adjoint_image and (nh > 0) rtm_offset_gather, downloads data_out, image
 * and gather.  Host buffers should be pinned for true asynchrony.  d_staging: caller-owned device
 * scratch of at least rtm_shot_staging_bytes(...) bytes.  Any output pointer may be NULL.         */
size_t rtm_shot_staging_bytes(const rtm_config *cfg, int nsrc, int nrec, int nh);
int rtm_shot_host(rtm_ctx *ctx, int nsrc, const float *h_src_xyz, const float *h_wav, int nrec,
                  const float *h_rec_xyz, const float *h_data_in, float *h_data_out, float scale,
                  float *h_image, int nh, const int *h_offsets, float *h_gather, void *d_staging,
                  size_t staging_bytes, void *cuda_stream);

/* ---- test hooks ------------------------------------------------------------------------------ */
/* Compressed wavefields in canonical order [r][N]: which = 0 Uz, 1 Vz.                            */
int rtm_export_probes(rtm_ctx *ctx, int which, float *d_out, void *cuda_stream);
/* Ask the NEXT pass to copy the wavefield(s) right after the listed steps (incl. injection) into
 * d_out [nsnap][nf][Np] canonical (nf = 1 acoustic, 2 TTI: p then r).  nsnap = 0 clears.          */
int rtm_set_snapshots(rtm_ctx *ctx, int nsnap, const int *h_steps, float *d_out);
/* Internal coefficient array in canonical [Np] order: which = 0 K2, 1 epsh, 2 delh, 3 cos, 4 sin (tilt), 5 cos, 6 sin
 * (azimuth, 3D TTI). */
int rtm_export_coeff(rtm_ctx *ctx, int which, float *d_out, void *cuda_stream);
/* Number of kernels this context has launched so far (bench.py's gpu_launches).                  */
long long rtm_launch_count(const rtm_ctx *ctx);
/* Device time [ms] of the step-kernel loop (nt launches, excluding the zero-fill and the final
 * sampling launch) of the last forward (which = 0) / adjoint (which = 1) pass, taken with CUDA events
 * on that pass's stream when option "time_steps" is 1.  Blocks the host until the pass has finished.
 * Negative if no timed pass has run.                                                               */
float rtm_last_pass_ms(rtm_ctx *ctx, int which);
/* The same, averaged over the last `count` (1..64) timed passes of that kind (bench.py: the mean launch duration over
 * the whole timed region, without a host synchronisation between shots).  Negative if fewer have run.      */
float rtm_pass_ms_mean(rtm_ctx *ctx, int which, int count);
/* Tuning knobs; none of them changes what is computed:
 *   "time_steps" 0|1  record CUDA events around the step launches of each pass (rtm_last_pass_ms);
 *   "pdl"        0|1  programmatic dependent launch between consecutive step kernels (default 1);
 *   "rx"         2|4|8|16|0  rows per thread of the 2D streaming kernel (0 = automatic; T > 1, 2D acoustic only);
 *   "resident"   0..3  2D acoustic with time-blocked probing: keep the wavefield in shared memory for a whole time block
 *                     (one launch per block instead of one per step).  1 (default): when the grid fits ONE thread-block
 *                     cluster (<= 16 slabs exchanging rows through distributed shared memory; small grids, which are
 *                     launch-bound otherwise); 2: beyond that also one slab per SM exchanging rows through L2 (measured
 *                     slower than the streaming kernel at c1); 3: the L2 mode only; 0: never.  Same bits
 *                     in every mode.
 *   "tti_tile"   16|32  2D TTI: rows per tile of the step kernel (256 or 512 threads per block).  32 (default when the time
 *                     block has 9 .. 16 steps, the only case it exists for) recomputes less halo; same bits either way.
 * Errors: RTM_EINVAL (unknown name / value out of range).
 * Timing experiments that break the results ("dbg" masks, per-block time stamps) exist only in a library built with
 * -DRTM_DEBUG (see the end of this header); the product build has neither.                                */
int rtm_set_option(rtm_ctx *ctx, const char *name, int value);

/* ---- the one entry point that allocates nothing ------------------------------------------------------------------
 * Offset gather (Eq. 4; reading C11) of caller-held compressed wavefields, for callers that cannot
 * allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): no context, no
 * workspace, no cudaMalloc / cudaFree / cudaMallocHost / event creation, no memcpy -- two kernel launches on `cuda_stream`
 * of the thread's CURRENT device and nothing else.
 *   gather[ih][x][z] = scale * sum_k U[k][x + h][z] V[k][x - h][z],  h = h_offsets[ih] grid points along x, zero where
 *   x + h or x - h leaves [0, nx);  h = 0 is Eq. 3's image.  2D grids.
 *   d_U, d_V   [r][nx][nz] fp32, DEVICE (the layout rtm_export_probes writes); read only
 *   h_offsets  [nh] HOST ints (passed to the device as a kernel argument: they may be reused when the call returns)
 *   d_gather   [nh][nx][nz] fp32, DEVICE, caller-owned; every element is written
 * Same arithmetic as rtm_offset_gather's generic kernel (the same gather_kernel: one fma per probe, k ascending), so
 * the two agree bit for bit on the same Uz / Vz.
 * Scratch: the kernel's operands -- U and V re-pitched to rows of 4 ceil(nz / 4) floats (16-byte loads) and the
 * offsets table -- live in ONE file-scope `static __device__` array of RTM_STATIC_SCRATCH_BYTES, which every GPU that
 * loads the library holds until the process exits.  Requests with
 *   256 + 2 * r * nx * 4 ceil(nz / 4) * 4 bytes > RTM_STATIC_SCRATCH_BYTES   or   nh > RTM_STATIC_MAX_OFFSETS
 * are rejected with RTM_ELIMIT before anything is launched.  Every call, on every stream and from every thread, shares
 * the array: it keeps the previous call's contents (each call rewrites all of what it reads, pad columns as zeros, so
 * nothing needs clearing by the caller), and two calls that overlap on the GPU (different streams without an ordering
 * between them) RACE on it.  Calls on one stream are ordered by the stream.
 * Errors: RTM_EINVAL (NULL, nx / nz / r / nh < 1, |h| >= nx), RTM_ELIMIT, RTM_ECUDA.                              */
#define RTM_STATIC_SCRATCH_BYTES (16u << 20)
#define RTM_STATIC_MAX_OFFSETS 64
#define RTM_ELIMIT (-5) /* size beyond the static scratch: RTM_STATIC_SCRATCH_BYTES / RTM_STATIC_MAX_OFFSETS */
int rtm_offset_gather_static(int nx, int nz, int r, const float *d_U, const float *d_V, int nh, const int *h_offsets,
                             float scale, float *d_gather, void *cuda_stream);

const char *rtm_strerror(int code);
const char *rtm_last_cuda_error(void);

#ifdef RTM_DEBUG
/* -DRTM_DEBUG builds only.  rtm_set_option(ctx, "dbg", mask): 1 no flush role, 2 no stencil role (RESULTS BECOME WRONG),
 * 16 write phase time stamps, 32 scalar arithmetic in the 3D streaming kernel (T = 16; bit-identical results).
 * rtm_debug_stamps: the first 8 phase time stamps (ns, %globaltimer) of each of the first nblocks (<= 1024) blocks of
 * the last step launch -> h_out [nblocks][8] (HOST).  Synchronises the device.                               */
int rtm_debug_stamps(rtm_ctx *ctx, unsigned long long *h_out, int nblocks);
#endif

#ifdef __cplusplus
}
#endif
#endif /* RTM_H */
