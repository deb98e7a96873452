// wd_handle.h — the handle behind include/wd.h and the helpers shared by the translation units that implement
// entry points (wd_api.cu, wd_gmres.cu, wd_dd.cu).  Not part of the C-ABI.
#pragma once
#include <string>

#include "../../include/wd.h"
#include "wd_internal.h"

static const int kMaxPipeChunks = 32;  // T chunks of the pipelined wd_apply_host (more chunks: shorter fill and drain)

using wd::MapCache;
struct wd_gmres_state;  // wd_gmres.cu
struct wd_dd_state;     // wd_dd.cu
struct wd_f32_state;    // wd_f32.cu

struct wd_handle {
    int n[4];
    long long V, Vs;  // sites; component stride of the device layout (elements)
    double m0, csw;
    int device;
    cudaStream_t stream;
    double2 *dU, *dS;
    double2 *dU2;          // two-row copy of the links (WD_OPT_GAUGE_ROWS = 2), or null
    unsigned int *dsched;  // work-queue words of the TMA kernels
    bool sched_dirty;      // a launch failed or the stream changed with work pending: re-zero the queue words first
    bool has_gauge, has_clover;
    bool clover_built;     // S was derived from the loaded links by wd_build_clover (a new gauge field invalidates it)
    int nsm;               // SMs of the handle's device
    MapCache *maps;        // tensor maps of the TMA kernels, keyed by (buffers, nrhs, tile)
    // options
    long variant, kernel_opt, tchunk_opt, zgroup_opt, device_pack, host_pipeline, gmres_graph, gauge_rows, f32_kernel;
    long rhs_block;  // WD_OPT_RHS_BLOCK: 1 = plain multi-RHS device layout, 4 = blocked (units of four interleaved per site)
    // staging
    double2 *pinned[2];
    size_t pinned_bytes;
    cudaEvent_t pinned_ev[2];
    double2 *dstage;
    size_t dstage_bytes;
    double2 *work_in, *work_out;  // wd_apply_host
    double2 *dstage_out;          // pipelined wd_apply_host: AoS staging of the result (a ring of chunks)
    size_t dstage_out_bytes;
    cudaStream_t s_up, s_dn;      // its upload and download streams
    cudaEvent_t ev_up[kMaxPipeChunks], ev_cmp[kMaxPipeChunks], ev_misc[2];
    bool pipe_ready;
    long launches;
    // config_epoch: bumped by everything that changes what a captured GMRES cycle has baked in (options, fields, the FP32
    // copies); fields_epoch: bumped when the FP64 links or S change — the FP32 copies remember the value they were made from
    long config_epoch, fields_epoch;
    std::string err;
    wd_gmres_state *gmres;  // workspace of wd_gmres (Krylov basis, Hessenberg matrix, CUDA graph), or null
    wd_dd_state *dd;        // sub-lattice state of a domain-decomposed operator (wd_create_local), or null
    wd_f32_state *f32;      // single-precision copies of the links and of S (wd_enable_f32), or null
};


namespace wd {

int fail(wd_handle *h, int code, const std::string &msg);  // records the text for wd_last_error, returns code

// Every entry point runs on the handle's device and leaves the caller's current device as it found it.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = (cudaSetDevice(dev) == cudaSuccess);
    }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
};
#define WD_ENTER(h) \
    if (!(h)) return WD_EINVAL; \
    wd::DeviceGuard guard_((h)->device)


// entry points that work on the plain device layout only
#define WD_PLAIN_ONLY(h, what) \
    if ((h)->rhs_block != 1) return wd::fail(h, WD_ESTATE, what ": not available while WD_OPT_RHS_BLOCK = 4 (blocked spinor layout)")

#define WD_CUDA(h, call)                                                                          \
    do {                                                                                          \
        cudaError_t e_ = (call);                                                                  \
        if (e_ != cudaSuccess)                                                                    \
            return wd::fail(h, (e_ == cudaErrorMemoryAllocation) ? WD_ENOMEM : WD_ECUDA,          \
                            std::string(#call) + ": " + cudaGetErrorString(e_));                 \
    } while (0)

// launch parameters of the handle's operator for kernel k (wd_api.cu)
int fill_params(wd_handle *h, KParams &p, const KernelInfo &k);
// one launch of a hopping / fused kernel on the handle's stream, with the work-queue and error bookkeeping
int launch_op(wd_handle *h, const KernelInfo &k, const KParams &p, int self);
void gmres_free(wd_handle *h);  // wd_gmres.cu
void dd_free(wd_handle *h);     // wd_dd.cu
void f32_free(wd_handle *h);    // wd_f32.cu
bool f32_current(const wd_handle *h);  // wd_f32.cu: FP32 copies exist and were made from the present FP64 fields
int dd_open_mask(const wd_handle *h);  // bit mu: direction mu does not wrap on this handle (wd_create_local)

}  // namespace wd
