/*
 * rflbm.h — C-ABI boundary of the B200-native D3Q27 regularized fluctuating lattice Boltzmann
 * (Reg-FLBM) collide-and-stream path of arXiv 2507.08820.
 *
 * Citations are PAPER.md line : equation.  "R<n>" are the readings listed in DESIGN.md.
 *
 * Conventions (all entry points)
 *   - Every function returns RFLBM_OK (0) or a negative code; none throws or aborts.  After a failure
 *     rflbm_last_error(h) returns a NUL-terminated description owned by the handle.
 *   - Pointers named *_dev are DEVICE pointers, *_host are HOST pointers.  The library NEVER allocates
 *     device memory and NEVER creates streams: the caller (PyTorch in this repository) owns both and
 *     must keep them alive for as long as the handle uses them (borrowed, never freed by the library).
 *   - Field layout: x fastest, site index s = x + nx*(y + ny*z); structure of arrays by component:
 *     rho[N], u[3][N], f[27][N] with N = nx*ny*nz.  Element type `real` = double (RFLBM_F64) or float
 *     (RFLBM_F32, fp32 population storage and fp32 arithmetic, R14).
 *   - Population order at the boundary ("canonical", R1): 0:(0,0,0); 1..6: +x,-x,+y,-y,+z,-z;
 *     7..10: (sx,sy,0); 11..14: (sx,0,sz); 15..18: (0,sy,sz) with (s1,s2) = (+,+),(+,-),(-,+),(-,-);
 *     19..26: (sx,sy,sz), sx outermost, sign order +,-.
 *   - Observable state (R10): the PRE-collision populations f_i(x,t) of Eq.1 after t steps;
 *     the internal storage (post-collision, un-streamed, A-B double buffer) is not exposed.
 *   - All work is enqueued on the stream given by rflbm_set_stream (default: the legacy stream 0) and is
 *     asynchronous unless stated otherwise.
 */
#ifndef RFLBM_H
#define RFLBM_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rflbm rflbm_t; /* opaque host-side handle */

enum { RFLBM_F64 = 0, RFLBM_F32 = 1 };
enum { RFLBM_OK = 0, RFLBM_EINVAL = -1, RFLBM_ESTATE = -2, RFLBM_ENOMEM = -3, RFLBM_ECUDA = -4 };

/* Problem definition: lattice size, hydrodynamic relaxation time tau_h = 1/omega_h (nu = (tau-1/2)/3,
 * PAPER.md:52; ghost rate omega_g = 1, :215), thermal energy kT (Eq.9 :99; kT = 0 -> deterministic
 * Reg-LBM, :294), reference density rho0 (:252), Philox seed (R8) and precision.
 * Host only: no GPU work, no allocation on the device.
 * EINVAL: nx,ny,nz < 1, N >= 2^32, nx > RFLBM_MAX_NX (27 padded rows must fit a 32-bit row offset), ny > 65535 *
 * max(1, 128/nx rounded down to a power of two) or nz > 65535 (launch grid limits), tau <= 0.5 or non-finite, kT < 0,
 * rho0 <= 0, unknown precision, out NULL. */
#define RFLBM_MAX_NX (2147483647 / 27 - 32) /* 79 536 399 */
int rflbm_create(int nx, int ny, int nz, double tau, double kT, double rho0, uint64_t seed, int precision,
                 rflbm_t** out);

/* Bytes of device workspace the handle needs: two population buffers of 27*px*ny*nzs*sizeof(real) bytes each (A-B
 * scheme; one for AA; px = nx rounded up to whole 128-byte lines for nx >= 32, nzs = nz, or nz+2 in slab mode), each
 * rounded up to 256 bytes, plus a 4 KiB reduction scratch and 12 KiB of Box-Muller tables. */
size_t rflbm_workspace_bytes(const rflbm_t* h);

/* Borrow `bytes` of device memory at dev_ptr (256-byte aligned) as the workspace.
 * ENOMEM if too small or misaligned.  Invalidates the state (rflbm_init / rflbm_set_populations needed).
 * The one call that writes to the device outside the handle's stream: it clears the 4 KiB scratch and uploads the
 * Box-Muller tables on the legacy stream and waits for both before returning (host-synchronous). */
int rflbm_set_workspace(rflbm_t* h, void* dev_ptr, size_t bytes);

/* cudaStream_t (as void*) on which every later call enqueues its work; borrowed. */
int rflbm_set_stream(rflbm_t* h, void* cuda_stream);

/* Solid layers z=0 and z=nz-1 with halfway bounce-back (R12; not in the paper, whose runs are periodic, :252).
 * Default off (periodic in x,y,z).  EINVAL if nz < 3.  Must be called before init/set_populations. */
int rflbm_set_walls_z(rflbm_t* h, int on);

/* Uniform acceleration g: body force F = rho*g, Guo forcing in moment form (R13).  Default 0. */
int rflbm_set_force(rflbm_t* h, double gx, double gy, double gz);

/* f = f^(0)(rho,u) (Eq.25 :225 with Eq.20 :160, R9); step counter := 0.
 * rho_dev = u_dev = NULL -> rho0, u = 0; else device arrays rho[N], u[3][N] of `real`.
 * ESTATE without a workspace. */
int rflbm_init(rflbm_t* h, const void* rho_dev, const void* u_dev);

/* Advance nsteps time steps of Eq.24 (:221): one fused pull-stream + collide kernel launch per step
 * (Eq.7 :87 pull form; Eq.2-3 :56-58; Eq.19 :153; Eq.20 :160; Eq.8-9 :93-99; Eq.10 :105).
 * rflbm_step(a); rflbm_step(b) is bit-identical to rflbm_step(a+b).  ESTATE before init. */
int rflbm_step(rflbm_t* h, int nsteps);

/* Storage scheme.  RFLBM_SCHEME_AB (default): two population buffers, read one / write the other.
 * RFLBM_SCHEME_AA: ONE buffer updated in place (half the footprint: 29 GB instead of 58 GB at 512^3 fp64, same
 * bytes moved per step): even steps read and write the site's own 27 slots (f*_q goes to slot 26-q), odd steps
 * read slot 26-q of x - c_q and write slot q of x + c_q; every thread writes exactly the locations it read.
 * Results are bit-identical to the A-B scheme (same arithmetic); the observable state (R10) does not depend on it.
 * Must be called before rflbm_set_workspace (ESTATE afterwards): rflbm_workspace_bytes depends on it. */
enum { RFLBM_SCHEME_AB = 0, RFLBM_SCHEME_AA = 1 };
int rflbm_set_scheme(rflbm_t* h, int scheme);

/* z-slab decomposition (PAPER.md:292 "the system was extended along the z direction", :300 "linear decomposition"):
 * this handle owns the nz layers [z0, z0+nz) of a GLOBAL lattice nx x ny x nz_global, periodic in z over nz_global.
 * The solid-layer test (walls at global z = 0 and nz_global-1) and the Philox site key x + nx (y + ny z) (R8) use the
 * global z, so the slabs together compute, bit for bit, what one handle of the undivided lattice computes.
 * The internal buffers get one ghost layer below and above; the faces travel through the four halo calls below,
 * which the CALLER moves between handles (cudaMemcpyAsync device-to-device, peer copy, NCCL/MPI send-recv ...): the
 * library itself never communicates.  In slab mode
 *   - the fields given to rflbm_init / rflbm_set_populations carry nz+2 layers: global layers z0-1 .. z0+nz
 *     (periodic in nz_global), i.e. rho[(nz+2)*ny*nx], u[3][...], f[27][...]; outputs have nz layers;
 *   - rflbm_step advances ONE step per call and, like the observables, fails with ESTATE while an exchange is
 *     pending (rflbm_halo_pending);
 *   - rflbm_run_host is not available.
 * Must be called before rflbm_set_workspace (ESTATE afterwards).  EINVAL: slab outside [0, nz_global), global lattice
 * with 2^32 sites or more, walls with nz_global < 3. */
int rflbm_set_slab(rflbm_t* h, int z0, int nz_global);

/* Face exchange of a slab.  Protocol, after rflbm_init / rflbm_set_populations and after every rflbm_step, with all
 * slabs at the same step count:
 *     if (rflbm_halo_pending(h)):   rflbm_halo_pack(h, LOW, a);  rflbm_halo_pack(h, HIGH, b);
 *                                   a -> the neighbour BELOW, which calls rflbm_halo_unpack(., HIGH, a)
 *                                   b -> the neighbour ABOVE, which calls rflbm_halo_unpack(., LOW,  b)
 * (periodic: the lowest slab's neighbour below is the highest slab).  A face buffer is 9 populations on one nx x ny
 * layer, packed [9][ny][nx] of `real`: rflbm_halo_bytes = 9*nx*ny*sizeof(real) (4.7 MB at 256^2 fp64).  What it
 * carries depends on the storage scheme and phase and is the library's business: the nine c_z = -1 (LOW) / c_z = +1
 * (HIGH) post-collision populations of the boundary layer that the neighbour will pull (A-B, and AA after an even
 * step), or, after an odd AA step, the nine populations this slab pushed across the face, which the neighbour takes
 * home into its own boundary layer.  pack and unpack enqueue one small kernel on the handle's stream and return;
 * they are no-ops (RFLBM_OK) when nothing is pending; a second rflbm_halo_unpack of a side that has
 * already been unpacked since the last step is a no-op too (the face is consumed once).  ESTATE: not in slab mode, or before init. */
enum { RFLBM_SIDE_LOW = 0, RFLBM_SIDE_HIGH = 1 };
size_t rflbm_halo_bytes(const rflbm_t* h);
int rflbm_halo_pending(const rflbm_t* h);
int rflbm_halo_pack(rflbm_t* h, int side, void* face_dev);
int rflbm_halo_unpack(rflbm_t* h, int side, const void* face_dev);

/* Ghost relaxation time tau_g = 1/omega_g of Reg-FLBM.  Default 1: the paper's final scheme, in
 * which the ghost part f^(1,g) drops out.  tau_g != 1 adds (1-omega_g) f^(1,g) with the recursive coefficients of
 * Eq.21 (:163-166, reading R20) and gives the ghost modes the noise amplitude of Eq.9 at omega_g.  Ignored by the
 * BGK model.  EINVAL: tau_g <= 0.5 or non-finite, or tau_g != 1 with a body force set. */
int rflbm_set_ghost_tau(rflbm_t* h, double tau_g);

/* Collision model.  RFLBM_MODEL_REG (default): the regularized fluctuating model, Eq.24, the hot
 * path.  RFLBM_MODEL_BGK: the paper's comparison model BGK-FLBM, Eq.11 (:109-111) with Eq.6 (:85): every
 * non-conserved mode k = 4..26 relaxes at the one rate omega = 1/tau and carries noise of amplitude Eq.9 at that
 * omega; f^eq is the Hermite equilibrium of Eq.25 (reading R19).  May be changed between steps (the state is the
 * populations).  EINVAL: unknown model, or BGK with a body force set (and rflbm_set_force refuses a non-zero
 * force while the model is BGK). */
enum { RFLBM_MODEL_REG = 0, RFLBM_MODEL_BGK = 1 };
int rflbm_set_model(rflbm_t* h, int model);

/* Which implementation of the step kernel rflbm_step launches.  AUTO (default): the TMA-staged kernel when kT > 0
 * and nx >= 32 (tiles of 128, 64 or 32 sites; the internal row pitch is padded so that any such nx qualifies), else
 * the plain one-thread-per-site kernel.  PLAIN forces the latter; TMA fails with EINVAL at rflbm_step if nx < 32.  All variants compute the same
 * update (same results up to the bit: identical arithmetic, only the data movement differs). */
enum { RFLBM_KERNEL_AUTO = 0, RFLBM_KERNEL_PLAIN = 1, RFLBM_KERNEL_TMA = 2 };
int rflbm_set_kernel_variant(rflbm_t* h, int variant);

/* rho[N], u[3][N] (device, `real`) of the current state: Eq.2-3, u = (j + F/2)/rho.  Solid nodes: 0. */
int rflbm_moments(rflbm_t* h, void* rho_dev, void* u_dev);

/* pi[6][N] (device, `real`): momentum-flux tensor Pi_ab = a_0,ab + a_1,ab = sum_i f_i (c_ia c_ib - delta_ab/3) of the
 * current state (Eq.18-19; the quantity the paper snapshots, :252, :260), order xx, yy, zz, xy, xz,
 * yz.  Solid nodes: 0. */
int rflbm_stress(rflbm_t* h, void* pi_dev);

/* The paper's snapshot (rho, rho u and Pi_ab saved every 5 000 steps) in ONE pass: rho[N], u[3][N] exactly
 * as rflbm_moments writes them and pi[6][N] exactly as rflbm_stress writes it (bit for bit), from a single gather of the
 * 27 populations: 27 reads + 10 writes per site (296 B at fp64) instead of 248 + 264 B for the two separate calls. */
int rflbm_snapshot(rflbm_t* h, void* rho_dev, void* u_dev, void* pi_dev);

/* Synchronises the stream.  out_host = { sum rho, sum rho u_x,y,z, mean u_x,y,z, var u_x,y,z } over fluid sites
 * (warp-shuffle + block reduction, fp64 accumulation).  A slab without a fluid site (one solid layer): all zeros. */
int rflbm_diagnostics(rflbm_t* h, double out_host[10]);

/* Canonical pre-collision populations f[27][N] (`real`, device) out of / into the handle.
 * set also sets the step counter (checkpoint/resume: the RNG is counter based, so resuming is bit exact). */
int rflbm_get_populations(rflbm_t* h, void* f_dev);
int rflbm_set_populations(rflbm_t* h, const void* f_dev, uint64_t step);

/* Test hook: what the step kernel draws at time `step` (R8): words[24][N] uint32 (6 Philox4x32-10 calls per
 * site, word 4q+m = output m of call q) and normals[23][N] `real` (modes k = 4..26).  Either may be NULL.
 * Synchronises the stream; ECUDA if the step kernel's hand-scheduled Philox rounds (csrc/rflbm_rng.cuh) disagree
 * with the plain ten-round loop at any site. */
int rflbm_debug_rng(rflbm_t* h, uint64_t step, void* words_dev, void* normals_dev);

/* End-to-end job with HOST buffers (what bench.py's "e2e" times): copy rho_host[N], u_host[3][N] (`real`,
 * pinned if the copies are to be asynchronous) to the device scratch, init, advance nsteps, compute moments, copy them
 * back to rho_out_host / u_out_host and synchronise.  scratch_dev: caller-owned device buffer of at least
 * 4*N*sizeof(real) bytes.  rho_host = u_host = NULL -> uniform rho0, u=0 start (no upload).
 * Afterwards the handle is in the state rflbm_init + rflbm_step(nsteps) leaves it in.
 * With a copy stream (rflbm_set_copy_stream) and the A-B scheme the job is PIPELINED, time-skewed along z: the fields are
 * uploaded in up to 32 bands of consecutive layers; as soon as the layers [0, U) are on the device, the state after L steps
 * is completed on the layers [L+1, U-1-L) for EVERY L (a step reaches one layer up and down, so each level runs one layer
 * behind the level below it), and the moments of the layers that have reached step nsteps are downloaded while the rest
 * is still being stepped (uploads and downloads share the copy stream and every upload is enqueued first, so the first
 * download starts once the last band is up); the triangular seam the periodic ring leaves open is closed at the end.  Jobs of
 * more than 24 steps skew only the first and the last 12 steps and run the steps in between as whole-lattice launches.
 * Every launch is the same kernel restricted to a z range, so the results are bit-identical to the serial form.
 * Without a copy stream, in the AA scheme, or with nz < 3, everything runs one after the other on the handle's stream.
 * ESTATE in slab mode.  ECUDA: a copy, event or launch failed (text of the FIRST failure in rflbm_last_error); both
 * streams are quiet when the call returns, and after a failed pipelined job the handle holds NO state (ESTATE until the
 * next rflbm_init / rflbm_set_populations / rflbm_run_host) and the output buffers are unspecified. */
int rflbm_run_host(rflbm_t* h, const void* rho_host, const void* u_host, int nsteps, void* rho_out_host,
                   void* u_out_host, void* scratch_dev, size_t scratch_bytes);

/* Test hook: the nth_call-th checked CUDA call (event, copy, wait, synchronise; counted from 1) of the NEXT pipelined
 * rflbm_run_host on this handle reports cudaErrorUnknown although it succeeded, so that the job's error path can be
 * exercised without corrupting the device; 0 disarms.  The job clears it when it returns. */
int rflbm_debug_inject_failure(rflbm_t* h, int nth_call);

/* A second cudaStream_t (as void*), borrowed, on which rflbm_run_host issues its host<->device copies so that they
 * overlap the kernels on the handle's stream (the two are ordered by events the call creates and destroys).
 * NULL (the default) or the handle's own stream: rflbm_run_host runs serially.  No other call uses it. */
int rflbm_set_copy_stream(rflbm_t* h, void* cuda_stream);

/* Number of kernels the handle has launched so far (bench.py's gpu_launches). */
uint64_t rflbm_launch_count(const rflbm_t* h);

/* Name of the step kernel the last rflbm_step launched ("step_kernel", "step_kernel_tma<TX=128>", ...; "" before the
 * first step): a static string, what bench.py reports as roofline.kernel. */
const char* rflbm_last_kernel(const rflbm_t* h);

/* The sums of rflbm_diagnostics for a caller that CANNOT ALLOCATE device memory: no handle, no workspace, nothing
 * allocated by the call (no cudaMalloc / cudaFree / allocating library routine, on the device or pinned).
 * rflbm_diagnostics itself needs a handle whose workspace holds one or two complete population buffers (29-58 GB at
 * 512^3 fp64).  A checkpoint inspector, an in-situ monitor or a plug-in that is handed a population field inside a
 * process whose device memory is already spoken for (the simulation owns the HBM, the host application owns the pool),
 * or that runs where cudaMalloc's device-wide synchronisation is not acceptable, has nowhere to get that from.  For
 * such callers the reduction scratch is part of the library image: a file-scope __device__ array of 2.5 MiB
 * (32 768 rows of 10 doubles + 1) that every GPU which loads librflbm.so carries until the process exits.
 *   f_dev      in   canonical PRE-collision populations f[27][N] (device, `real` by `precision`; what
 *                   rflbm_get_populations writes), N = nx*ny*nz, x fastest.  Borrowed for the duration of the call.
 *   walls_z    in   non-zero: layers z = 0 and z = nz-1 are solid and excluded (R12); needs nz >= 3
 *   g_host     in   acceleration g[3] (host) or NULL for none: the reported velocity is u = j/rho + g/2 (R13)
 *   stream     in   cudaStream_t (as void*) on the CURRENT device; f_dev must live on the current device
 *   out_host   out  { sum rho, sum rho u_x,y,z, mean u_x,y,z, var u_x,y,z } over the fluid sites, as rflbm_diagnostics
 *   err_host   out  optional (may be NULL): err_len bytes that receive a NUL-terminated message on failure
 * Limit: N <= rflbm_static_max_sites() = RFLBM_STATIC_MAX_SITES = 2^27 (512^3, the headline lattice).  Anything larger
 * is refused with RFLBM_EINVAL and a message naming the limit, before any GPU work.  Other EINVAL: NULL f_dev /
 * out_host, sizes < 1, unknown precision, non-finite g, f_dev not device memory of the current device.  ECUDA: a CUDA
 * call failed.
 * The call enqueues two kernels and an 80-byte copy on `stream` and waits for the stream (host-synchronous, like
 * rflbm_diagnostics).  No atomics: repeated calls on the same field return the same bits.
 * First call on a device: looks up the device address of the static array (cudaGetSymbolAddress, cached per device);
 * with the runtime's lazy module loading this is also the moment the array and the two kernels take their device
 * memory.  Make that first call outside any stream capture.
 * Sharing: all calls on one GPU, from any thread or handle, use the same array, and it keeps what the last call left in
 * it.  Nothing in it needs to start at zero (every row a call reads it has written itself first), but two calls that
 * overlap on the GPU (different streams, different threads) race on it and return garbage: serialise them. */
#define RFLBM_STATIC_MAX_SITES 134217728LL
long long rflbm_static_max_sites(void);
int rflbm_diagnostics_static(const void* f_dev, int nx, int ny, int nz, int precision, int walls_z, const double* g_host,
                             void* cuda_stream, double out_host[10], char* err_host, size_t err_len);

uint64_t rflbm_step_count(const rflbm_t* h);
const char* rflbm_last_error(const rflbm_t* h);

/* Frees the host handle only (the workspace belongs to the caller). */
int rflbm_destroy(rflbm_t* h);

#ifdef __cplusplus
}
#endif
#endif /* RFLBM_H */
