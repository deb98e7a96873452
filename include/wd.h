/* include/wd.h — C-ABI of libwd: the finest-level Wilson(-clover) Dirac operator on one B200.
 *
 *   (D psi)(x) = S(x) psi(x)
 *              - 1/2 sum_mu [ (I4 - gamma_mu) (x) U_mu(x)       ] psi(x + mu)
 *              - 1/2 sum_mu [ (I4 + gamma_mu) (x) U_mu(x - mu)^H ] psi(x - mu)        (eq. 1.13,
 *   S(x) = (m0+4) I12 - csw/32 sum_{mu,nu} (gamma_mu gamma_nu) (x) (Q_mu_nu(x) - Q_nu_mu(x))
 *                                                      PAPER.md:227-230; eq. 2.5)
 * with lattice spacing a = 1, periodic boundary conditions in all four directions
 * (PAPER.md:187), FP64 complex arithmetic, and the gamma matrices of DESIGN.md R1.
 *
 * Plain C: opaque handle, plain pointers (each documented as HOST or DEVICE) and sizes, no torch
 * or C++ types.  Every function returns 0 (WD_OK) or a negative error code; nothing throws or
 * aborts across this boundary; wd_last_error() gives the text of the last failure on a handle.
 *
 * CANONICAL HOST LAYOUTS (what the paper's CPU code stores; complex = re,im):
 *   site index      i = ((t*Z + z)*Y + y)*X + x, 0-based, X fastest; V = T*Z*Y*X
 *   directions      mu = 0,1,2,3 = T,Z,Y,X
 *   spinor          double [nrhs][V][12][2], component 3*spin + colour
 *   gauge           double [V][4][3][3][2]: forward links U_mu(x) of the own site, row-major 3x3
 *
 *   self-coupling   double [V][42][2]: the 42 entries of S(x) = D_sc, INCLUDING the
 *                   (m0+4) diagonal: entries 0..11 the real diagonal (imaginary part ignored),
 *                   12..26 the strict upper triangle, row-major, of S[0:6,0:6] (spins 0,1),
 *                   27..41 the same of S[6:12,6:12] (spins 2,3); lower triangles are the
 *                   conjugates (R6).
 *
 * DEVICE LAYOUT: chosen by the library, opaque to the caller.
 * A device spinor buffer holds wd_spinor_bytes(h, nrhs) bytes, is at least 16-byte aligned (checked;
 * cudaMalloc and PyTorch give 256 bytes or more), and is filled / read with wd_pack_spinor /
 * wd_unpack_spinor (or wd_apply_host).  Fields stay
 * device-resident in device layout between applications: wd_apply never repacks (the lesson of
 * PAPER.md:1015, where per-application reordering ate the gain).
 *
 * OWNERSHIP: the library owns gauge, self-coupling and staging storage on the device; the
 * caller owns every pointer it passes in (host arrays are copied before the call returns;
 * device spinor buffers are caller-allocated, e.g. by PyTorch).
 *
 * THREADING: a handle is used by one host thread at a time.  All device work of a handle is
 * issued on the handle's stream (default: the legacy default stream; see wd_set_stream).
 *
 * DEVICE: a handle belongs to the CUDA device that was current in wd_create.  Every entry point
 * switches to that device for the duration of the call and restores the caller's current device.
 */
#ifndef WD_H
#define WD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct wd_handle wd_handle;

enum {
    WD_OK = 0,
    WD_EINVAL = -1, /* bad dimensions, null pointer, nrhs < 1, unknown option or value         */
    WD_ENOMEM = -2, /* host or device allocation failed                                          */
    WD_ESTATE = -3, /* e.g. apply before the gauge field is loaded, clover missing with csw != 0 */
    WD_ECUDA = -4   /* a CUDA runtime call or kernel launch failed (text in wd_last_error)       */
};

/* Options for wd_set_option / wd_get_option. */
enum {
    WD_OPT_VARIANT = 1,   /* 0 = fused single pass (default), 1 = unfused: hopping kernel + self-coupling kernel */
    WD_OPT_KERNEL = 2,    /* hopping/fused kernel geometry id; -1 = automatic (default); see wd_kernel_name        */
    WD_OPT_TCHUNK = 3,    /* T-extent marched by one CTA in tiled geometries; 0 = automatic                       */
    WD_OPT_ZGROUP = 4,    /* number of Z-tiles per rasterisation group in tiled geometries; 0 = automatic         */
    WD_OPT_DEVICE_PACK = 5,/* 1 = wd_load_* / wd_pack_* transpose on the device instead of on the host (default 0) */
    WD_OPT_HOST_PIPELINE = 6,/* wd_apply_host: 1 = overlap upload, compute and download over T chunks (default), 0 = serial */
    WD_OPT_GMRES_GRAPH = 7,/* wd_gmres: 1 = replay restart cycles as one CUDA graph (default; needs a non-default stream), 0 = launch by launch.
                              A captured cycle is reused only for the same x, b, m, tol and stream AND an unchanged handle: any
                              wd_set_option, wd_load_gauge, wd_load_clover, wd_build_clover or wd_enable_f32 makes the next solve capture anew */
    WD_OPT_GAUGE_ROWS = 8  /* 3 = links stored as 9 complex numbers (default).  2 = two-row storage for SU(3) links: the
                              fused TMA kernel of one right-hand side reads rows 0, 1 (384 instead of 576 B per site) and
                              rebuilds row 2 = conj(row 0 x row 1) in registers.  EXACT ONLY FOR SU(3) LINKS: with 2 the
                              "general 3x3 complex" promise of wd_load_gauge (R11) does not hold.  Costs a second,
                              two-row copy of the gauge field on the device. */
    ,WD_OPT_F32_KERNEL = 9 /* wd_apply_f32: 0 = automatic (the TMA kernel where its 2x4x16 tile divides the lattice), 1 = always
                              the one-thread-per-site kernels */
    ,WD_OPT_RHS_BLOCK = 10 /* Device layout of spinor buffers that hold SEVERAL right-hand sides ("multi-tuple" storage, cf.
                              PAPER.md:15, :1037).  1 (default): plain, double2 [nrhs][12][Vs].  4: BLOCKED, double2
                              [ceil(nrhs/4)][12][Vs][4] — the right-hand sides of a unit of four interleaved per site, the last
                              unit padded to four — the layout of the fastest multi-RHS kernel (tmqb_*: every spinor access of
                              a warp is 512 consecutive bytes, the links and S of a site are read once for its four right-hand
                              sides).  Changes what wd_spinor_bytes / wd_pack_spinor / wd_unpack_spinor / wd_apply mean by a
                              device spinor buffer, for every nrhs; set it before allocating buffers.  Needs a lattice the
                              2x4x8 tile divides (else WD_EINVAL).  While it is 4, wd_apply_host, wd_gmres, the wd_dd_* and the
                              *_f32 calls and the unfused variant return WD_ESTATE (they use the plain layout). */
};

/* Create an operator for a T x Z x Y x X periodic lattice.  Every extent >= 1 (n = 2, where
 * x+mu and x-mu are the same site, and n = 1 are handled: both hopping terms are applied,
 * DESIGN.md R12).  csw == 0: pure Wilson, S = (m0+4) I, no self-coupling array is needed.
 * csw != 0: S must be supplied with wd_load_clover or built with wd_build_clover.
 * Uses the current CUDA device.  Errors: WD_EINVAL, WD_ENOMEM, WD_ECUDA. */
int wd_create(wd_handle **h, int T, int Z, int Y, int X, double m0, double csw);

/* Free all device and host storage of the handle.  Synchronises the handle's stream. */
int wd_destroy(wd_handle *h);

/* HOST pointer, canonical gauge layout.  Packed into the device layout and copied; the caller
 * keeps ownership.  Links are treated as general 3x3 complex matrices (U and U^H are used,
 * never U^-1; R11).  Synchronous w.r.t. the host array.
 * A self-coupling field that wd_build_clover derived from the PREVIOUS links is discarded: with
 * csw != 0 the next wd_apply returns WD_ESTATE until wd_build_clover or wd_load_clover is called
 * again.  A field supplied with wd_load_clover is the caller's and is kept. */
int wd_load_gauge(wd_handle *h, const double *host_U);

/* HOST pointer, canonical self-coupling layout (the whole S(x), eq. 2.5).  Required iff csw != 0
 * (allowed also with csw == 0: the loaded S then replaces (m0+4) I). */
int wd_load_clover(wd_handle *h, const double *host_C);

/* Build S(x) of eq. 2.5 on the device from the loaded gauge field (Q_mu_nu of eq. 1.12,
 * PAPER.md:221, all 16 ordered pairs, R8) with the handle's m0 and csw.
 * Errors: WD_ESTATE if no gauge field is loaded. */
int wd_build_clover(wd_handle *h);

/* Read S(x) back: HOST pointer, canonical self-coupling layout [V][42][2]. */
int wd_get_clover(wd_handle *h, double *host_C);

/* out = D in for nrhs right-hand sides (eq. 1.13).  DEVICE pointers in DEVICE layout, each
 * wd_spinor_bytes(h, nrhs) bytes, 16-byte aligned; out must not overlap in.  Asynchronous:
 * enqueued on the handle's stream, no host synchronisation, no host<->device copies, no
 * repacking.  Errors: WD_EINVAL, WD_ESTATE (no gauge; csw != 0 and no self-coupling), WD_ECUDA. */
int wd_apply(wd_handle *h, void *dev_out, const void *dev_in, int nrhs);

/* Restarted GMRES(m) with right preconditioning M = I for D x = b (Algorithm 1 of the paper, PAPER.md:240-289;
 * modified Gram-Schmidt, h_ij = v_i^H w, R16), entirely on the device: the operator is wd_apply, the
 * orthogonalisation, norms, the (m+1) x m least-squares problem and the solution update are kernels of this library
 * that keep every scalar in device memory.  dev_x: DEVICE spinor (device layout, one right-hand side), the initial
 * guess x_0 on entry and the approximate solution on return; dev_b: DEVICE spinor, not modified; 1 <= m <= 64.
 * Termination (R17): ||b - D x|| < tol * ||b - D x_0||, tested on the true residual at the top
 * of every restart cycle, or max_cycles cycles done; inside a cycle |h_{j+1,j}| < tol / 10 ends the Arnoldi loop
 * (R18).  *cycles_done (may be NULL) = cycles performed; host_resid (HOST, may be NULL, max_cycles + 1
 * doubles): host_resid[k] = ||b - D x|| after k cycles.  The library owns (m + 2) work spinors, kept for the next
 * call.  Synchronises the handle's stream once per cycle (to read the residual norm); with a non-default stream the
 * second and later cycles are one CUDA graph launch each (WD_OPT_GMRES_GRAPH).
 * Errors: WD_EINVAL, WD_ESTATE (no gauge / no self-coupling field), WD_ENOMEM, WD_ECUDA. */
int wd_gmres(wd_handle *h, void *dev_x, const void *dev_b, int m, int max_cycles, double tol, int *cycles_done,
             double *host_resid);

/* The same algorithm in MIXED precision (SURVEY.md section 8(f)3 + 8(f)4; the paper's operator exists in both precisions,
 * PAPER.md:642): the Krylov vectors v_1 .. v_{m+1}, the operator applications w = D v_j (wd_apply_f32) and the
 * orthogonalisation run on single-precision vectors; the residual r = b - D x of line 4 (wd_apply), the solution x,
 * every inner product, norm and entry of H are double.  Each restart cycle is thus a defect correction: it solves
 * D e = r approximately in single precision and adds e to the double-precision x, so the iteration converges to the
 * solution of the DOUBLE-precision system as long as a cycle reduces the residual at all (single precision limits the
 * reduction per cycle to about 1e-6, not the final accuracy).  Arguments, termination and errors as wd_gmres; dev_x
 * and dev_b are FP64 device spinors.  Needs wd_enable_f32 (WD_ESTATE otherwise).  The library owns (m + 2)
 * single-precision work spinors and one double-precision one.  CUDA graph as wd_gmres. */
int wd_gmres_mixed(wd_handle *h, void *dev_x, const void *dev_b, int m, int max_cycles, double tol, int *cycles_done,
                   double *host_resid);

/* The Hessenberg matrix of the LAST restart cycle of the last wd_gmres call as the Arnoldi process produced it:
 * host_H (HOST, may be NULL): (m+1) * m complex numbers, column-major with leading dimension m + 1
 * (host_H[2 * (i + (m+1) * j)] = Re h_{i+1,j+1}); *kdim (may be NULL) = Krylov dimension of that cycle (m unless the
 * breakdown rule ended it); *lsq_resid (may be NULL) = min_y ||beta e_1 - H y||, the recurrence residual. */
int wd_gmres_last_hessenberg(wd_handle *h, double *host_H, int *kdim, double *lsq_resid);

/* ---- an entry point that allocates nothing ----
 * WHO IT IS FOR.  Every other call of this library may reach cudaMalloc: wd_create and the wd_load_ / wd_enable_ calls
 * always do, wd_gmres does for its Krylov basis and for the partial sums and counters of its reductions.  Some programs
 * cannot afford that at the point where they need an inner product or a norm of device spinors: a solver written on top of
 * PyTorch (or any framework whose caching allocator has already taken nearly all of the 180 GB), where a raw cudaMalloc
 * from a library fails or carves memory out behind the allocator's back; an iteration loop between two operator
 * applications, where cudaMalloc / cudaFree would stall every stream of the device because they synchronise it; a host
 * program that forbids driver allocations after its own start-up phase.  For them:
 *
 * wd_inner_product_static: dev_result[r] = <a_r, b_r> = sum over the 12 components and the V sites of conj(a) * b, for
 * r = 0 .. nrhs-1 — h_ij = v_i^H w of Algorithm 1 lines 10-11 and, with dev_a == dev_b, the squared norms of lines 5
 * and 14.  No handle: dev_a, dev_b are DEVICE spinors of the current device in the PLAIN device layout
 * (complex double [nrhs][12][Vs], of which the first V elements of every component are read; V = sites,
 * Vs = wd_component_stride), dev_result is a DEVICE array of nrhs complex doubles; all three caller-owned and 16-byte
 * aligned; cuda_stream as in wd_set_stream.  Asynchronous on that stream.  Same kernel structure and, for nrhs = 1, the
 * same summation order as the reductions inside wd_gmres, so the result is deterministic.
 *
 * SCRATCH.  The per-block partial sums and the completion counters of the reduction sit in ONE fixed array of 65 792 bytes
 * (4096 partial sums + 64 counters) that is part of the library image: every GPU on which libwd.so is loaded holds it from
 * load to process exit, whether or not this function is ever called, and it never grows.  LIMIT: nrhs <= 64 per call (one
 * counter per right-hand side); a larger nrhs is refused with WD_EINVAL and a text that says so — split the call.  V is
 * not limited by the scratch (blocks loop over the sites).
 *
 * FIRST CALL ON A DEVICE.  The first call made with a given device current asks the CUDA runtime once for the address the
 * array has on that device and keeps it (no allocation, but a runtime query that is not stream work): make that first call
 * during set-up, before any stream capture is begun on that device; later calls only enqueue a 256-byte memset of the
 * counters and one kernel.
 *
 * SHARING.  All calls on a device, from every stream and thread, use the same array, and it keeps what the previous call
 * left in it.  The function clears the counters itself on every call; the partial sums need no clearing (each block writes
 * its slot before any is read).  Two calls whose GPU work can overlap — different streams without an event between them,
 * or two host threads — race on the array and return garbage: order them yourself.  Calls on one stream are safe.
 *
 * Errors: WD_EINVAL (null or misaligned pointer, V < 1, Vs < V, nrhs < 1, nrhs > 64), WD_ECUDA; text in
 * wd_last_error(NULL).  Never WD_ENOMEM. */
int wd_inner_product_static(const void *dev_a, const void *dev_b, long long V, long long Vs, int nrhs, void *dev_result,
                            void *cuda_stream);

/* ---- domain decomposition (Algorithm 3; local lattices, eqs. 2.1-2.4) ----
 * A handle for ONE hyper-rectangular sub-lattice of a global periodic lattice: local extents = global_dims / proc_grid
 * (int[4] each, order T,Z,Y,X; proc_coords = position of this sub-lattice in the grid).  In a direction with
 * proc_grid[mu] > 1 ("decomposed") the local lattice does not wrap: wd_apply on such a handle computes everything that
 * needs no neighbour — the hops across the two faces of that direction are left out — and wd_dd_exterior adds them from
 * the half-spinors the neighbours packed with wd_dd_pack.  Gauge field: the forward links of the LOCAL sites only
 * (wd_load_gauge, local canonical layout); no ghost links exist.  Self-coupling: wd_load_clover (S of the local sites,
 * computed from the global field); wd_build_clover returns WD_ESTATE on a decomposed handle (plaquettes cross the seam).
 * One application:   wd_dd_pack (every decomposed mu)  ->  exchange of the buffers by the caller (NCCL / peer / device
 * copies), overlapping with  wd_apply  ->  wd_dd_exterior (every decomposed mu), all on the handle's stream. */
int wd_create_local(wd_handle **h, const int *global_dims, const int *proc_grid, const int *proc_coords, double m0,
                    double csw);

/* Bit mu set: direction mu is decomposed on this handle (0 for a handle made by wd_create). */
int wd_dd_open_mask(const wd_handle *h);

/* Sites of one face of direction mu (V / n_mu) and bytes of one face buffer, nrhs * 6 * face_sites * 16; 0 if mu is not
 * decomposed.  Face sites are enumerated in canonical order of the three remaining coordinates (X fastest), the same
 * on both sides of a seam; a buffer is complex double [nrhs][6][face_sites]. */
long long wd_dd_face_sites(const wd_handle *h, int mu);
size_t wd_dd_face_bytes(const wd_handle *h, int mu, int nrhs);

/* Alg. 3 lines 1-16 for direction mu.  dev_in: DEVICE spinor(s) in device layout.  Writes (DEVICE buffers of
 * wd_dd_face_bytes each, caller-allocated):
 *   dev_send_minus: lambda_mu(x) = rows 0,1 of (I4 - gamma_mu) psi(x), x on the low face — goes to the -mu neighbour,
 *                   which passes it to wd_dd_exterior as dev_recv_from_plus;
 *   dev_send_plus:  rows 0,1 of (I4 + gamma_mu) (x) U_mu(x)^H psi(x), x on the high face — goes to the +mu neighbour
 *                   as its dev_recv_from_minus.   (The factor 1/2 of Alg. 3 is applied in wd_dd_exterior.) */
int wd_dd_pack(wd_handle *h, const void *dev_in, int nrhs, int mu, void *dev_send_minus, void *dev_send_plus);

/* Alg. 3 lines 17-31 for direction mu: dev_out (the result of wd_apply on this handle, same stream) receives
 * -1/2 (I4 - gamma_mu) (x) U_mu(x) lambda on the high face and -1/2 times the (I4 + gamma_mu)-reconstruction of chi on
 * the low face. */
int wd_dd_exterior(wd_handle *h, void *dev_out, int nrhs, int mu, const void *dev_recv_from_plus,
                   const void *dev_recv_from_minus);

/* ---- FP32 variant (the paper's PRECISION templating) ----
 * wd_enable_f32: makes single-precision copies of the loaded links and of S on the device.  The copies go stale when the
 * FP64 fields change (wd_load_gauge, wd_load_clover, wd_build_clover): wd_apply_f32 and wd_gmres_mixed then return
 * WD_ESTATE until wd_enable_f32 is called again.  A single-precision device spinor is the device layout with 8-byte elements: wd_spinor_bytes_f32
 * bytes, 8-byte aligned; it is produced from / turned into an FP64 device spinor by wd_convert_spinor (to_f32 = 1:
 * dst float <- src double; 0: dst double <- src float; both DEVICE pointers).  wd_apply_f32: out = D in with every load,
 * store and arithmetic operation in FP32 (one fused pass per right-hand side); the error against the FP64 operator is
 * bounded in DESIGN.md ("Tolerance of the FP32 variant": relative L2 <= 1e-6).  Asynchronous on the handle's stream.
 * Errors: WD_ESTATE (fields missing / wd_enable_f32 not called), WD_EINVAL, WD_ENOMEM, WD_ECUDA. */
int wd_enable_f32(wd_handle *h);
size_t wd_spinor_bytes_f32(const wd_handle *h, int nrhs);
int wd_convert_spinor(wd_handle *h, void *dev_dst, const void *dev_src, int nrhs, int to_f32);
int wd_apply_f32(wd_handle *h, void *dev_out, const void *dev_in, int nrhs);

/* Same operation on HOST arrays in canonical spinor layout: host->device copy, on-device
 * repack, operator, repack, device->host copy, all inside the call; returns after the result is
 * in host_out.  With a TMA kernel the lattice is cut into up to 32 chunks along T and upload,
 * compute and download of different chunks overlap on three streams (the library's own two plus
 * the handle's); otherwise the steps run one after the other on the handle's stream.  Pinned
 * host memory lets the copies overlap and is faster, but is not required.  Result identical bit
 * for bit to wd_pack_spinor / wd_apply / wd_unpack_spinor. */
int wd_apply_host(wd_handle *h, double *host_out, const double *host_in, int nrhs);

/* Size in bytes of a device spinor buffer for nrhs right-hand sides (0 on error).  It is
 * nrhs * 12 * wd_component_stride(h) * 16 — a little more than nrhs * V * 192, see below; with
 * WD_OPT_RHS_BLOCK = 4, nrhs is rounded up to a multiple of four first. */
size_t wd_spinor_bytes(const wd_handle *h, int nrhs);

/* Component stride Vs of the device layout, in complex elements (0 on error): component c of
 * right-hand side r of a device spinor starts at element (12*r + c) * Vs and holds the V sites in
 * canonical order, followed by Vs - V elements of padding that are never read or written.  The
 * padding keeps the components of one site from aliasing onto one L2 slice when V*16 B is a
 * power of two. */
long long wd_component_stride(const wd_handle *h);
/* Blocked multi-RHS layout (WD_OPT_RHS_BLOCK = 4): right-hand sides 4u .. 4u+3 form unit u; element (c, site i, r) of
 * unit u is at complex element ((12*u + c) * Vs + i) * 4 + r of the buffer.  A unit occupies the same 4 * 12 * Vs elements
 * as four right-hand sides of the plain layout, so "right-hand sides 4u onwards" start at the same offset in both.  The
 * slots of a last, partial unit are zero-filled by wd_pack_spinor and hold unspecified values after wd_apply. */

/* HOST canonical [nrhs][V][12][2]  <->  DEVICE layout.  Synchronous. */
int wd_pack_spinor(wd_handle *h, void *dev_dst, const double *host_src, int nrhs);
int wd_unpack_spinor(wd_handle *h, double *host_dst, const void *dev_src, int nrhs);

/* The host packer by itself (step a0; no GPU needed): writes the host-side IMAGE of the device
 * layout of one field — exactly the bytes wd_load_gauge / wd_load_clover / wd_pack_spinor place
 * in device memory — and its inverse.  field: WD_FIELD_SPINOR (one RHS, canonical 12 complex per
 * site), WD_FIELD_GAUGE (36), WD_FIELD_CLOVER (canonical 42 complex -> 36 packed slots; unpacking
 * returns zero imaginary parts on the diagonal), WD_FIELD_SPINOR_BLOCK4 (one unit of the blocked multi-RHS layout:
 * canonical [4][nsites][12] -> [12][nsites][4], the image wd_pack_spinor writes with WD_OPT_RHS_BLOCK = 4).  HOST
 * pointers; nsites = V.  wd_layout_bytes: size of the packed image (0 on error). */
enum { WD_FIELD_SPINOR = 0, WD_FIELD_GAUGE = 1, WD_FIELD_CLOVER = 2, WD_FIELD_SPINOR_BLOCK4 = 3 };
size_t wd_layout_bytes(int field, long long nsites);
int wd_layout_pack_host(int field, long long nsites, const double *canonical, double *packed);
int wd_layout_unpack_host(int field, long long nsites, const double *packed, double *canonical);

/* cudaStream_t passed as void* (NULL = legacy default stream).  PyTorch supplies memory and
 * streams only.  Waits for the work already enqueued on the previous stream (the handle's work
 * queue and staging buffers are shared by all its launches). */
int wd_set_stream(wd_handle *h, void *cuda_stream);

/* Block the host until all work enqueued on the handle's stream has finished. */
int wd_synchronize(wd_handle *h);

int wd_set_option(wd_handle *h, int option, long value);
int wd_get_option(const wd_handle *h, int option, long *value);

/* Number of compiled kernel geometries and their names ("linear256", "tile_1x4x4x16", ...);
 * NULL if id is out of range.  wd_kernel_in_use: the id the next wd_apply will launch. */
int wd_kernel_count(void);
const char *wd_kernel_name(int id);
int wd_kernel_in_use(const wd_handle *h);
/* The kernel wd_apply(h, ..., nrhs) launches (the automatic choice depends on whether there is a clover term and on
 * whether several right-hand sides are applied in one call); wd_kernel_in_use(h) = wd_kernel_for(h, 1). */
int wd_kernel_for(const wd_handle *h, int nrhs);

/* Number of kernel launches issued by this handle so far (all kernels of this library). */
long wd_launch_count(const wd_handle *h);

/* Text of the last error on this handle (h == NULL: of the last failed wd_create or handle-free call on this thread).
 * Never NULL. */
const char *wd_last_error(const wd_handle *h);

const char *wd_version(void);

#ifdef __cplusplus
}
#endif
#endif /* WD_H */
