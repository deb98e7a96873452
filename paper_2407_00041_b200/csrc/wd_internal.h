// wd_internal.h — shared declarations of libwd's translation units (not part of the C-ABI).
#pragma once
#include <cuda_runtime.h>

#include <string>

namespace wd {

// ---------------------------------------------------------------------------------------------
// Device layout ("SoA over sites").  Element = one complex
// double = double2 = 16 B; the site index i (canonical order, X fastest) is the fastest index of
// every array, so a warp that handles 32 consecutive sites reads 512 contiguous bytes per
// component:
// The component stride is Vs = V rounded up to 16 sites + 272 sites of padding (component_stride()): every
// component starts 256-byte aligned and the components of one site are not a power of two apart.  Measured
// at 64^4 (profiles/r1b_*.md): padding of 0 .. 16400 sites all within 1 % — kept because it is free.
//   spinor  double2 [nrhs][12][Vs]      component c = 3*spin + colour
//   gauge   double2 [4][9][Vs]          mu = T,Z,Y,X; k = 3*row + col; forward links only, each
//                                       link stored ONCE (U_mu(x-mu) is read from site x-mu)
//   selfcpl double2 [36][Vs]            18 slots per chirality block b (A = 0, B = 1), block-contiguous
//                                       so that one block is one TMA box: slot 18b+j (j<3) holds the
//                                       real diagonal pair (B_{2j,2j}, B_{2j+1,2j+1}); slot 18b+3+k the
//                                       k-th strict-upper entry (row-major) of the 6x6 block
//                                       (72 reals = 576 B per site, R6/R7)
// ---------------------------------------------------------------------------------------------
long long component_stride(long long V);  // wd_api.cu

constexpr int kSpinorComps = 12;
constexpr int kGaugeComps = 36;
constexpr int kCloverSlots = 36;
constexpr int kCloverCanon = 42;

__host__ __device__ constexpr int slot_diag(int b, int j) { return 18 * b + j; }      // j = 0..2
__host__ __device__ constexpr int slot_off(int b, int k) { return 18 * b + 3 + k; }   // k = 0..14

enum SelfMode { SELF_NONE = 0, SELF_MASS = 1, SELF_CLOVER = 2 };

struct MapCache;  // wd_tma_common.cuh: per-handle cache of tensor maps

struct KParams {
    const double2 *psi;  // right-hand side 0; RHS r at + r * 12 * Vs (same for out)
    int nrhs;            // right-hand sides of this launch (> 1 only for kernels with multi_rhs)
    const double2 *U;
    const double2 *U2;   // two-row copy of the links, double2 [4][6][Vs] (rows 0 and 1), or null
    const double2 *S;
    double2 *out;
    long long V;    // sites
    long long Vs;   // component stride in elements (V plus padding, see component_stride())
    int n[4];       // T, Z, Y, X
    int stride[4];  // site-index strides of T, Z, Y, X
    double mass;    // m0 + 4
    // tiled geometries: rasterisation of CTAs (see wd_kernels.cu)
    int ntx, nty, ntz, ntc;  // number of tiles in X, Y, Z and of T-chunks
    int gz;                  // Z-tiles per rasterisation group
    int tchunk;              // T-extent marched by one CTA
    int opt_tchunk, opt_zgroup;  // the raw WD_OPT_TCHUNK / WD_OPT_ZGROUP values (0 = automatic)
    unsigned int *sched;         // device, 2 words, zero between launches: work queue of the TMA kernels
    int tc_begin, tc_count;      // TMA kernels: apply only to T chunks [tc_begin, tc_begin + tc_count) of opt_tchunk
                                 // slices each (tc_count = 0: the whole lattice); used by the pipelined wd_apply_host
    int nsm, device;             // SM count and ordinal of the handle's device (read once in wd_create)
    MapCache *maps;              // tensor-map cache of the handle (may be null: encode per launch)
    int open_mask;               // bit mu: direction mu does not wrap (sub-lattice of a domain decomposition, wd_dd.cu)
    int esize;                   // bytes per complex element of the fields: 16 (FP64), 8 (FP32 variant: the pointers above are float2)
    int gauge_rows;              // 3: links stored as 9 complex; 2: two-row storage, third row rebuilt in the kernel
};

struct KernelInfo {
    const char *name;
    int bt, bz, by, bx;  // tile extents (all 0: linear geometry, any lattice)
    int threads;
    bool multi_rhs;      // one launch applies the operator to all p.nrhs right-hand sides
    int rhs_block;       // device layout of the spinors it reads and writes: 1 plain, 4 blocked (WD_OPT_RHS_BLOCK)
    cudaError_t (*launch)(const KParams &p, int self, cudaStream_t st);
};

int kernel_count();
const KernelInfo &kernel_info(int id);

// TMA-staged T-marching kernels: first generation (wd_tma.cu), second generation (wd_tmb.cu)
cudaError_t launch_tma_2x4x16(const KParams &p, int self, cudaStream_t st);
cudaError_t launch_tmq_2x4x8(const KParams &p, int self, cudaStream_t st);   // four right-hand sides per work item
cudaError_t launch_tmqb_2x4x8(const KParams &p, int self, cudaStream_t st);  // the same on the blocked multi-RHS layout
cudaError_t launch_tmb_4x4x8(const KParams &p, int self, cudaStream_t st);
cudaError_t launch_tmb_2x4x16(const KParams &p, int self, cudaStream_t st);  // three ring slots
// first generation with two compute warpgroups per tile (wd_tmw.cu)
cudaError_t launch_tmw_2x4x16(const KParams &p, int self, cudaStream_t st);
MapCache *map_cache_new();
void map_cache_delete(MapCache *c);
void map_cache_clear(MapCache *c);

// self-coupling kernel of the unfused variant: out += S psi (clover) or out += mass * psi
cudaError_t launch_selfcoupling(const KParams &p, int self, cudaStream_t st);

// device-side layout transposes (wd_pack.cu): canonical AoS <-> device SoA (component stride Vs)
cudaError_t launch_aos_to_soa(double2 *dst_soa, const double2 *src_aos, long long V, long long Vs, int ncomp, cudaStream_t st);
cudaError_t launch_soa_to_aos(double2 *dst_aos, const double2 *src_soa, long long V, long long Vs, int ncomp, cudaStream_t st);
cudaError_t launch_clover_canon_to_dev(double2 *dst_slots, const double2 *src42, long long V, long long Vs, cudaStream_t st);
cudaError_t launch_clover_dev_to_canon(double2 *dst42, const double2 *src_slots, long long V, long long Vs, cudaStream_t st);

// host packers (wd_pack.cu): canonical AoS chunk [i0, i0+cnt) -> SoA staging [ncomp][cnt]
void host_pack_aos_to_soa(double2 *dst, const double2 *src_aos, long long i0, long long cnt, int ncomp);
void host_unpack_soa_to_aos(double2 *dst_aos, const double2 *src, long long i0, long long cnt, int ncomp);
void host_pack_clover(double2 *dst, const double2 *src42, long long i0, long long cnt);
void host_unpack_clover(double2 *dst42, const double2 *src, long long i0, long long cnt);
// blocked multi-RHS layout, one unit of B right-hand sides: staging [12][cnt][B] <-> canonical spinors src[r] (each
// [V][12]) rows i0 .. i0+cnt; right-hand sides r >= nlive are written as zeros / not read back
void host_pack_spinor_blocked(double2 *dst, const double2 *const *src, int B, int nlive, long long i0, long long cnt);
void host_unpack_spinor_blocked(double2 *const *dst, const double2 *src, int B, int nlive, long long i0, long long cnt);

// two-row copy of the gauge field (wd_pack.cu): U2[mu][k] = U[mu][k], k = 0..5
cudaError_t launch_compress_gauge(double2 *U2, const double2 *U, long long V, long long Vs, cudaStream_t st);

// device clover construction (wd_clover.cu): S slots from the device gauge field
cudaError_t launch_build_clover(double2 *S_slots, const double2 *U, const int n[4], long long V, long long Vs,
                                double mass, double csw, cudaStream_t st);

}  // namespace wd
