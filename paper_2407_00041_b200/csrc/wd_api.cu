// wd_api.cu — the C-ABI of include/wd.h: handle, storage, load/pack paths, kernel selection.
// There is no CPU fallback anywhere in this library: every operator application is a kernel
// launch; if CUDA is unavailable the calls fail with WD_ECUDA.
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>

#include "wd_handle.h"

using namespace wd;

static thread_local std::string g_create_err = "";

// Component stride of the device SoA layout.  V rounded up to 16 sites (256 B, keeps every component
// 256-byte aligned for TMA / 128-bit access) plus 17 * 16 sites, so that consecutive components differ
// in the low address bits that select the L2 slice and set (measured: no effect on B200; kept
// because it is free).  With -DWD_EXPERIMENTS, WD_PAD_SITES overrides the padding (any multiple of 16 >= 0).
long long wd::component_stride(long long V) {
    long long pad = 16 * 17;
#ifdef WD_EXPERIMENTS
    if (const char *e = getenv("WD_PAD_SITES")) {
        const long long v = atoll(e);
        if (v >= 0 && v % 16 == 0) pad = v;
    }
#endif
    return (V + 15) / 16 * 16 + pad;
}

int wd::fail(wd_handle *h, int code, const std::string &msg) {
    if (h) h->err = msg; else g_create_err = msg;
    return code;
}

static const size_t kStageSites = 1 << 16;  // sites per host staging chunk

static int ensure_pinned(wd_handle *h, size_t bytes) {
    if (h->pinned_bytes >= bytes) return WD_OK;
    for (int b = 0; b < 2; b++) {
        if (h->pinned[b]) cudaFreeHost(h->pinned[b]);
        h->pinned[b] = nullptr;
    }
    h->pinned_bytes = 0;
    for (int b = 0; b < 2; b++) WD_CUDA(h, cudaMallocHost((void **)&h->pinned[b], bytes));
    h->pinned_bytes = bytes;
    return WD_OK;
}

static int ensure_dstage(wd_handle *h, size_t bytes) {
    if (h->dstage_bytes >= bytes) return WD_OK;
    if (h->dstage) cudaFree(h->dstage);
    h->dstage = nullptr;
    h->dstage_bytes = 0;
    WD_CUDA(h, cudaMalloc((void **)&h->dstage, bytes));
    h->dstage_bytes = bytes;
    return WD_OK;
}

static void release_dstage(wd_handle *h) {
    if (h->dstage) cudaFree(h->dstage);
    h->dstage = nullptr;
    h->dstage_bytes = 0;
}

// (re)build the two-row copy of the links when two-row storage is selected and a gauge field is present
static int refresh_two_row_copy(wd_handle *h) {
    if (h->gauge_rows != 2 || !h->has_gauge) return WD_OK;
    if (!h->dU2) WD_CUDA(h, cudaMalloc((void **)&h->dU2, (size_t)h->Vs * 24 * sizeof(double2)));
    WD_CUDA(h, launch_compress_gauge(h->dU2, h->dU, h->V, h->Vs, h->stream));
    h->launches++;
    map_cache_clear(h->maps);
    return WD_OK;
}

extern "C" {

const char *wd_version(void) { return "wd-b200 0.2 (sm_100a; FP64, FP32 variant)"; }

const char *wd_last_error(const wd_handle *h) { return h ? h->err.c_str() : g_create_err.c_str(); }

int wd_create(wd_handle **out, int T, int Z, int Y, int X, double m0, double csw) {
    if (!out) return fail(nullptr, WD_EINVAL, "wd_create: null handle pointer");
    *out = nullptr;
    if (T < 1 || Z < 1 || Y < 1 || X < 1) return fail(nullptr, WD_EINVAL, "wd_create: every lattice extent must be >= 1");
    const long long V = (long long)T * Z * Y * X;
    // site indices are 64-bit everywhere; a T slice (the stride of T) must fit an int, the whole field the device
    if ((long long)Z * Y * X >= (1LL << 31) || V >= (1LL << 40)) return fail(nullptr, WD_EINVAL, "wd_create: lattice too large");
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(nullptr, WD_ECUDA, std::string("wd_create: no CUDA device: ") + cudaGetErrorString(e));
    wd_handle *h = new (std::nothrow) wd_handle();
    if (!h) return fail(nullptr, WD_ENOMEM, "wd_create: out of host memory");
    h->n[0] = T; h->n[1] = Z; h->n[2] = Y; h->n[3] = X;
    h->V = V;
    h->Vs = component_stride(V);
    h->m0 = m0;
    h->csw = csw;
    h->device = dev;
    h->stream = nullptr;
    h->dU = h->dS = h->dU2 = nullptr;
    h->dsched = nullptr;
    h->sched_dirty = false;
    h->has_gauge = h->has_clover = h->clover_built = false;
    h->nsm = 148;
    if (cudaDeviceGetAttribute(&h->nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || h->nsm < 1) h->nsm = 148;
    h->maps = map_cache_new();
    h->host_pipeline = 1;
    h->gmres_graph = 1;
    h->gauge_rows = 3;
    h->f32_kernel = 0;
    h->rhs_block = 1;
    h->variant = 0;
    h->kernel_opt = -1;
    h->tchunk_opt = 0;
    h->zgroup_opt = 0;
    h->device_pack = 0;
    h->pinned[0] = h->pinned[1] = nullptr;
    h->pinned_bytes = 0;
    h->pinned_ev[0] = h->pinned_ev[1] = nullptr;
    h->dstage = nullptr;
    h->dstage_bytes = 0;
    h->work_in = h->work_out = nullptr;
    h->dstage_out = nullptr;
    h->dstage_out_bytes = 0;
    h->s_up = h->s_dn = nullptr;
    h->pipe_ready = false;
    h->launches = 0;
    h->config_epoch = h->fields_epoch = 0;
    h->gmres = nullptr;
    h->dd = nullptr;
    h->f32 = nullptr;
    e = cudaMalloc((void **)&h->dU, (size_t)h->Vs * kGaugeComps * sizeof(double2));
    if (e == cudaSuccess) e = cudaMalloc((void **)&h->dsched, 2 * sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaMemset(h->dsched, 0, 2 * sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->pinned_ev[0], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->pinned_ev[1], cudaEventDisableTiming);
    if (e != cudaSuccess) {
        const int code = (e == cudaErrorMemoryAllocation) ? WD_ENOMEM : WD_ECUDA;
        fail(nullptr, code, std::string("wd_create: ") + cudaGetErrorString(e));
        wd_destroy(h);
        cudaGetLastError();
        return code;
    }
    *out = h;
    return WD_OK;
}

int wd_destroy(wd_handle *h) {
    WD_ENTER(h);
    cudaStreamSynchronize(h->stream);
    gmres_free(h);
    dd_free(h);
    f32_free(h);
    map_cache_delete(h->maps);
    if (h->dU) cudaFree(h->dU);
    if (h->dS) cudaFree(h->dS);
    if (h->dU2) cudaFree(h->dU2);
    if (h->dsched) cudaFree(h->dsched);
    if (h->dstage) cudaFree(h->dstage);
    if (h->work_in) cudaFree(h->work_in);
    if (h->work_out) cudaFree(h->work_out);
    if (h->dstage_out) cudaFree(h->dstage_out);
    if (h->pipe_ready) {
        cudaStreamDestroy(h->s_up);
        cudaStreamDestroy(h->s_dn);
        for (int k = 0; k < kMaxPipeChunks; k++) {
            cudaEventDestroy(h->ev_up[k]);
            cudaEventDestroy(h->ev_cmp[k]);
        }
        cudaEventDestroy(h->ev_misc[0]);
        cudaEventDestroy(h->ev_misc[1]);
    }
    for (int b = 0; b < 2; b++) {
        if (h->pinned[b]) cudaFreeHost(h->pinned[b]);
        if (h->pinned_ev[b]) cudaEventDestroy(h->pinned_ev[b]);
    }
    delete h;
    return WD_OK;
}

int wd_set_stream(wd_handle *h, void *cuda_stream) {
    WD_ENTER(h);
    if ((cudaStream_t)cuda_stream == h->stream) return WD_OK;
    // work pending on the old stream still uses the handle's work queue and staging: let it finish first
    WD_CUDA(h, cudaStreamSynchronize(h->stream));
    h->stream = (cudaStream_t)cuda_stream;
    return WD_OK;
}

int wd_synchronize(wd_handle *h) {
    WD_ENTER(h);
    WD_CUDA(h, cudaStreamSynchronize(h->stream));
    return WD_OK;
}

// ---- host -> device loads ---------------------------------------------------------------------
// Generic chunked path: pack `cnt` sites into pinned staging [ncomp_dev][cnt], then one strided
// 2-D copy into the SoA arrays (row pitch V elements).  Two staging buffers alternate so that
// packing chunk k+1 overlaps the copy of chunk k.
typedef void (*pack_fn)(double2 *, const double2 *, long long, long long);

static void pack_gauge_chunk(double2 *dst, const double2 *src, long long i0, long long cnt) {
    host_pack_aos_to_soa(dst, src, i0, cnt, kGaugeComps);
}
static void pack_spinor_chunk(double2 *dst, const double2 *src, long long i0, long long cnt) {
    host_pack_aos_to_soa(dst, src, i0, cnt, kSpinorComps);
}

static int load_chunked(wd_handle *h, double2 *dev, const double2 *host, int ncomp_dev, pack_fn pack) {
    const long long V = h->V;
    const long long chunk = (V < (long long)kStageSites) ? V : (long long)kStageSites;
    int rc = ensure_pinned(h, (size_t)chunk * 42 * sizeof(double2));
    if (rc) return rc;
    int b = 0;
    for (long long i0 = 0; i0 < V; i0 += chunk, b ^= 1) {
        const long long cnt = (V - i0 < chunk) ? V - i0 : chunk;
        WD_CUDA(h, cudaEventSynchronize(h->pinned_ev[b]));
        pack(h->pinned[b], host, i0, cnt);
        WD_CUDA(h, cudaMemcpy2DAsync(dev + i0, (size_t)h->Vs * sizeof(double2), h->pinned[b], (size_t)cnt * sizeof(double2),
                                     (size_t)cnt * sizeof(double2), ncomp_dev, cudaMemcpyHostToDevice, h->stream));
        WD_CUDA(h, cudaEventRecord(h->pinned_ev[b], h->stream));
    }
    WD_CUDA(h, cudaStreamSynchronize(h->stream));
    return WD_OK;
}

typedef void (*unpack_fn)(double2 *, const double2 *, long long, long long);
static void unpack_spinor_chunk(double2 *dst, const double2 *src, long long i0, long long cnt) {
    host_unpack_soa_to_aos(dst, src, i0, cnt, kSpinorComps);
}

static int store_chunked(wd_handle *h, double2 *host, const double2 *dev, int ncomp_dev, unpack_fn unpack) {
    const long long V = h->V;
    const long long chunk = (V < (long long)kStageSites) ? V : (long long)kStageSites;
    int rc = ensure_pinned(h, (size_t)chunk * 42 * sizeof(double2));
    if (rc) return rc;
    for (long long i0 = 0; i0 < V; i0 += chunk) {
        const long long cnt = (V - i0 < chunk) ? V - i0 : chunk;
        WD_CUDA(h, cudaMemcpy2DAsync(h->pinned[0], (size_t)cnt * sizeof(double2), dev + i0, (size_t)h->Vs * sizeof(double2),
                                     (size_t)cnt * sizeof(double2), ncomp_dev, cudaMemcpyDeviceToHost, h->stream));
        WD_CUDA(h, cudaStreamSynchronize(h->stream));
        unpack(host, h->pinned[0], i0, cnt);
    }
    return WD_OK;
}

int wd_load_gauge(wd_handle *h, const double *host_U) {
    WD_ENTER(h);
    if (!host_U) return fail(h, WD_EINVAL, "wd_load_gauge: null pointer");
    h->config_epoch++, h->fields_epoch++;
    if (h->clover_built) {  // S was built from the links that are being replaced: it must be rebuilt (or loaded)
        h->has_clover = h->clover_built = false;
    }
    h->has_gauge = false;
    const size_t bytes = (size_t)h->V * kGaugeComps * sizeof(double2);
    if (h->device_pack) {
        int rc = ensure_dstage(h, bytes);
        if (rc) return rc;
        WD_CUDA(h, cudaMemcpyAsync(h->dstage, host_U, bytes, cudaMemcpyHostToDevice, h->stream));
        WD_CUDA(h, launch_aos_to_soa(h->dU, h->dstage, h->V, h->Vs, kGaugeComps, h->stream));
        h->launches++;
        WD_CUDA(h, cudaStreamSynchronize(h->stream));
        release_dstage(h);
    } else {
        int rc = load_chunked(h, h->dU, (const double2 *)host_U, kGaugeComps, pack_gauge_chunk);
        if (rc) return rc;
    }
    h->has_gauge = true;
    return refresh_two_row_copy(h);
}

static int ensure_clover_storage(wd_handle *h) {
    if (!h->dS) WD_CUDA(h, cudaMalloc((void **)&h->dS, (size_t)h->Vs * kCloverSlots * sizeof(double2)));
    return WD_OK;
}

int wd_load_clover(wd_handle *h, const double *host_C) {
    WD_ENTER(h);
    if (!host_C) return fail(h, WD_EINVAL, "wd_load_clover: null pointer");
    h->config_epoch++, h->fields_epoch++;
    int rc = ensure_clover_storage(h);
    if (rc) return rc;
    if (h->device_pack) {
        const size_t bytes = (size_t)h->V * kCloverCanon * sizeof(double2);
        rc = ensure_dstage(h, bytes);
        if (rc) return rc;
        WD_CUDA(h, cudaMemcpyAsync(h->dstage, host_C, bytes, cudaMemcpyHostToDevice, h->stream));
        WD_CUDA(h, launch_clover_canon_to_dev(h->dS, h->dstage, h->V, h->Vs, h->stream));
        h->launches++;
        WD_CUDA(h, cudaStreamSynchronize(h->stream));
        release_dstage(h);
    } else {
        rc = load_chunked(h, h->dS, (const double2 *)host_C, kCloverSlots, host_pack_clover);
        if (rc) return rc;
    }
    h->has_clover = true;
    h->clover_built = false;
    return WD_OK;
}

int wd_build_clover(wd_handle *h) {
    WD_ENTER(h);
    if (!h->has_gauge) return fail(h, WD_ESTATE, "wd_build_clover: no gauge field loaded");
    if (dd_open_mask(h))
        return fail(h, WD_ESTATE, "wd_build_clover: plaquettes cross the seams of a decomposed handle; load S with wd_load_clover");
    h->config_epoch++, h->fields_epoch++;
    int rc = ensure_clover_storage(h);
    if (rc) return rc;
    WD_CUDA(h, launch_build_clover(h->dS, h->dU, h->n, h->V, h->Vs, h->m0 + 4.0, h->csw, h->stream));
    h->launches++;
    h->has_clover = true;
    h->clover_built = true;
    return WD_OK;
}

int wd_get_clover(wd_handle *h, double *host_C) {
    WD_ENTER(h);
    if (!host_C) return fail(h, WD_EINVAL, "wd_get_clover: null pointer");
    if (!h->has_clover) return fail(h, WD_ESTATE, "wd_get_clover: no self-coupling field present");
    return store_chunked(h, (double2 *)host_C, h->dS, kCloverSlots, host_unpack_clover);
}

// ---- spinors ------------------------------------------------------------------------------------
size_t wd_spinor_bytes(const wd_handle *h, int nrhs) {
    if (!h || nrhs < 1) return 0;
    const size_t slots = (h->rhs_block > 1) ? (size_t)((nrhs + h->rhs_block - 1) / h->rhs_block * h->rhs_block) : (size_t)nrhs;
    return slots * (size_t)h->Vs * kSpinorComps * sizeof(double2);
}

// Blocked multi-RHS layout (WD_OPT_RHS_BLOCK = B): unit u = right-hand sides uB .. uB+B-1 is double2 [12][Vs][B].  Seen as
// a field of 12 components whose "sites" are B elements wide, a chunk of sites is one strided 2-D copy like the plain layout.
// Staging [12][cnt][B]; right-hand sides past the last one are zero.
static int pack_spinor_blocked(wd_handle *h, double2 *dev, const double2 *host, int nrhs) {
    const long long V = h->V, B = h->rhs_block;
    const long long chunk = (V < (long long)kStageSites) ? V : (long long)kStageSites;
    int rc = ensure_pinned(h, (size_t)chunk * kSpinorComps * B * sizeof(double2));
    if (rc) return rc;
    const size_t per = (size_t)V * kSpinorComps, uper = (size_t)h->Vs * kSpinorComps * B;
    int b = 0;
    for (int u = 0; u * B < nrhs; u++)
        for (long long i0 = 0; i0 < V; i0 += chunk, b ^= 1) {
            const long long cnt = (V - i0 < chunk) ? V - i0 : chunk;
            WD_CUDA(h, cudaEventSynchronize(h->pinned_ev[b]));
            double2 *st = h->pinned[b];
            const double2 *src[8];
            const int nlive = (nrhs - u * B < B) ? (int)(nrhs - u * B) : (int)B;
            for (int r = 0; r < B; r++) src[r] = host + (size_t)(u * B + (r < nlive ? r : 0)) * per;
            host_pack_spinor_blocked(st, src, (int)B, nlive, i0, cnt);
            WD_CUDA(h, cudaMemcpy2DAsync(dev + u * uper + i0 * B, (size_t)h->Vs * B * sizeof(double2), st, (size_t)cnt * B * sizeof(double2),
                                         (size_t)cnt * B * sizeof(double2), kSpinorComps, cudaMemcpyHostToDevice, h->stream));
            WD_CUDA(h, cudaEventRecord(h->pinned_ev[b], h->stream));
        }
    WD_CUDA(h, cudaStreamSynchronize(h->stream));
    return WD_OK;
}

static int unpack_spinor_blocked(wd_handle *h, double2 *host, const double2 *dev, int nrhs) {
    const long long V = h->V, B = h->rhs_block;
    const long long chunk = (V < (long long)kStageSites) ? V : (long long)kStageSites;
    int rc = ensure_pinned(h, (size_t)chunk * kSpinorComps * B * sizeof(double2));
    if (rc) return rc;
    const size_t per = (size_t)V * kSpinorComps, uper = (size_t)h->Vs * kSpinorComps * B;
    for (int u = 0; u * B < nrhs; u++)
        for (long long i0 = 0; i0 < V; i0 += chunk) {
            const long long cnt = (V - i0 < chunk) ? V - i0 : chunk;
            double2 *st = h->pinned[0];
            WD_CUDA(h, cudaMemcpy2DAsync(st, (size_t)cnt * B * sizeof(double2), dev + u * uper + i0 * B, (size_t)h->Vs * B * sizeof(double2),
                                         (size_t)cnt * B * sizeof(double2), kSpinorComps, cudaMemcpyDeviceToHost, h->stream));
            WD_CUDA(h, cudaStreamSynchronize(h->stream));
            double2 *dst[8];
            const int nlive = (nrhs - u * B < B) ? (int)(nrhs - u * B) : (int)B;
            for (int r = 0; r < B; r++) dst[r] = host + (size_t)(u * B + (r < nlive ? r : 0)) * per;
            host_unpack_spinor_blocked(dst, st, (int)B, nlive, i0, cnt);
        }
    return WD_OK;
}

long long wd_component_stride(const wd_handle *h) { return h ? h->Vs : 0; }

static bool misaligned(const void *p) { return ((size_t)p & 15) != 0; }

int wd_pack_spinor(wd_handle *h, void *dev_dst, const double *host_src, int nrhs) {
    WD_ENTER(h);
    if (!dev_dst || !host_src || nrhs < 1 || misaligned(dev_dst)) return fail(h, WD_EINVAL, "wd_pack_spinor: bad argument");
    if (h->rhs_block > 1) return pack_spinor_blocked(h, (double2 *)dev_dst, (const double2 *)host_src, nrhs);
    const size_t per = (size_t)h->V * kSpinorComps, dper = (size_t)h->Vs * kSpinorComps;
    for (int r = 0; r < nrhs; r++) {
        double2 *dst = (double2 *)dev_dst + r * dper;
        const double2 *src = (const double2 *)host_src + r * per;
        if (h->device_pack) {
            int rc = ensure_dstage(h, per * sizeof(double2));
            if (rc) return rc;
            WD_CUDA(h, cudaMemcpyAsync(h->dstage, src, per * sizeof(double2), cudaMemcpyHostToDevice, h->stream));
            WD_CUDA(h, launch_aos_to_soa(dst, h->dstage, h->V, h->Vs, kSpinorComps, h->stream));
            h->launches++;
            WD_CUDA(h, cudaStreamSynchronize(h->stream));
        } else {
            int rc = load_chunked(h, dst, src, kSpinorComps, pack_spinor_chunk);
            if (rc) return rc;
        }
    }
    return WD_OK;
}

int wd_unpack_spinor(wd_handle *h, double *host_dst, const void *dev_src, int nrhs) {
    WD_ENTER(h);
    if (!host_dst || !dev_src || nrhs < 1 || misaligned(dev_src)) return fail(h, WD_EINVAL, "wd_unpack_spinor: bad argument");
    if (h->rhs_block > 1) return unpack_spinor_blocked(h, (double2 *)host_dst, (const double2 *)dev_src, nrhs);
    const size_t per = (size_t)h->V * kSpinorComps, dper = (size_t)h->Vs * kSpinorComps;
    for (int r = 0; r < nrhs; r++) {
        double2 *dst = (double2 *)host_dst + r * per;
        const double2 *src = (const double2 *)dev_src + r * dper;
        if (h->device_pack) {
            int rc = ensure_dstage(h, per * sizeof(double2));
            if (rc) return rc;
            WD_CUDA(h, launch_soa_to_aos(h->dstage, src, h->V, h->Vs, kSpinorComps, h->stream));
            h->launches++;
            WD_CUDA(h, cudaMemcpyAsync(dst, h->dstage, per * sizeof(double2), cudaMemcpyDeviceToHost, h->stream));
            WD_CUDA(h, cudaStreamSynchronize(h->stream));
        } else {
            int rc = store_chunked(h, dst, src, kSpinorComps, unpack_spinor_chunk);
            if (rc) return rc;
        }
    }
    return WD_OK;
}

// ---- the host packer alone (CPU-testable) -------------------------------------------------------
size_t wd_layout_bytes(int field, long long nsites) {
    if (nsites < 1) return 0;
    switch (field) {
    case WD_FIELD_SPINOR: return (size_t)nsites * kSpinorComps * sizeof(double2);
    case WD_FIELD_GAUGE: return (size_t)nsites * kGaugeComps * sizeof(double2);
    case WD_FIELD_CLOVER: return (size_t)nsites * kCloverSlots * sizeof(double2);
    case WD_FIELD_SPINOR_BLOCK4: return (size_t)nsites * kSpinorComps * 4 * sizeof(double2);
    default: return 0;
    }
}

int wd_layout_pack_host(int field, long long nsites, const double *canonical, double *packed) {
    if (nsites < 1 || !canonical || !packed) return WD_EINVAL;
    switch (field) {
    case WD_FIELD_SPINOR: host_pack_aos_to_soa((double2 *)packed, (const double2 *)canonical, 0, nsites, kSpinorComps); return WD_OK;
    case WD_FIELD_GAUGE: host_pack_aos_to_soa((double2 *)packed, (const double2 *)canonical, 0, nsites, kGaugeComps); return WD_OK;
    case WD_FIELD_CLOVER: host_pack_clover((double2 *)packed, (const double2 *)canonical, 0, nsites); return WD_OK;
    case WD_FIELD_SPINOR_BLOCK4: {
        const double2 *src[4];
        for (int r = 0; r < 4; r++) src[r] = (const double2 *)canonical + (size_t)r * nsites * kSpinorComps;
        host_pack_spinor_blocked((double2 *)packed, src, 4, 4, 0, nsites);
        return WD_OK;
    }
    default: return WD_EINVAL;
    }
}

int wd_layout_unpack_host(int field, long long nsites, const double *packed, double *canonical) {
    if (nsites < 1 || !canonical || !packed) return WD_EINVAL;
    switch (field) {
    case WD_FIELD_SPINOR: host_unpack_soa_to_aos((double2 *)canonical, (const double2 *)packed, 0, nsites, kSpinorComps); return WD_OK;
    case WD_FIELD_GAUGE: host_unpack_soa_to_aos((double2 *)canonical, (const double2 *)packed, 0, nsites, kGaugeComps); return WD_OK;
    case WD_FIELD_CLOVER: host_unpack_clover((double2 *)canonical, (const double2 *)packed, 0, nsites); return WD_OK;
    case WD_FIELD_SPINOR_BLOCK4: {
        double2 *dst[4];
        for (int r = 0; r < 4; r++) dst[r] = (double2 *)canonical + (size_t)r * nsites * kSpinorComps;
        host_unpack_spinor_blocked(dst, (const double2 *)packed, 4, 4, 0, nsites);
        return WD_OK;
    }
    default: return WD_EINVAL;
    }
}

// ---- kernel selection -----------------------------------------------------------------------------
static bool geometry_fits(const wd_handle *h, const KernelInfo &k) {
    if (k.bx == 0) return true;
    return h->n[0] % k.bt == 0 && h->n[1] % k.bz == 0 && h->n[2] % k.by == 0 && h->n[3] % k.bx == 0;
}

static int auto_kernel(const wd_handle *h, int nrhs) {
    // Preference order.  One right-hand side with a clover term, fused: the warpgroup-split
    // kernel (64^4: 4.13 ms burst / 4.30 ms sustained against 4.15 / 4.35 ms of the first generation, which stays the
    // choice with two-row links).  The hopping term alone (csw = 0, or the unfused variant): the second generation on
    // the 2x4x16 tile (pure Wilson 2.75 ms; 4x4x8 tile 2.88, tmw 3.06, tma 3.66 ms).  Several right-hand sides in one
    // call: the quad kernels of wd_tmq.cu (cfg 5: tmqb on the blocked layout 17.4 ms, tmq on the plain layout 20.8 ms when
    // its units of four are well filled), else the second generation on the 4x4x8 tile with its four-slot ring (25.4 ms;
    // 2x4x16 with three slots 28.3, tmw 27.4, tma 28.5 ms).  linear256 always fits, and wins on small lattices.
    static const char *pref_clover[] = {"tmw_2x4x16", "tma_2x4x16", "tmb_4x4x8"};
    static const char *pref_tworow[] = {"tma_2x4x16", "tmw_2x4x16", "tmb_4x4x8"};
    static const char *pref_hop[] = {"tmb_2x4x16", "tmb_4x4x8", "tmw_2x4x16"};
    static const char *pref_multi[] = {"tmb_4x4x8", "tmb_2x4x16", "tmw_2x4x16"};
    if (h->rhs_block > 1) {  // blocked multi-RHS layout: the kernels written for it
        for (int id = 0; id < kernel_count(); id++)
            if (kernel_info(id).rhs_block == h->rhs_block && geometry_fits(h, kernel_info(id))) return id;
        return 0;
    }
    // several right-hand sides on the plain layout: the quad kernel when its units of four are well filled (cfg 5: 21.7 ms
    // against 26.4 ms of tmb_4x4x8; a unit costs the same however many of its four right-hand sides exist)
    if (nrhs > 1 && h->variant == 0 && 20 * nrhs >= 17 * 4 * ((nrhs + 3) / 4))
        for (int id = 0; id < kernel_count(); id++)
            if (!strcmp(kernel_info(id).name, "tmq_2x4x8") && geometry_fits(h, kernel_info(id))) return id;
    // small lattices: a persistent TMA kernel costs ~25 us to start and drain whatever the volume; below 32 Ki sites the
    // one-thread-per-site kernel wins for one or two right-hand sides (8^4: 13 us against 31 us; 8x8x16x32: 14.5 against
    // 16.9 us; 16^4: 37 against 24.5 us, so not beyond)
    if (h->V <= 32768 && nrhs <= 2) return 0;  // linear256
    const bool clover_fused = (h->csw != 0.0 || h->has_clover) && h->variant == 0;
    const char **pref = (nrhs > 1 && h->variant == 0) ? pref_multi : !clover_fused ? pref_hop : (h->gauge_rows == 2) ? pref_tworow : pref_clover;
    // (the tiled one-thread-per-site kernels are never chosen: linear256 beats them wherever no TMA tile divides the
    // lattice — 20^4: 88 against 113 us, 36^4: 0.80 against 1.04 ms — they stay selectable with WD_OPT_KERNEL)
    for (int i = 0; i < 3; i++)
        for (int id = 0; id < kernel_count(); id++)
            if (!strcmp(kernel_info(id).name, pref[i]) && geometry_fits(h, kernel_info(id))) return id;
    return 0;
}

int wd_kernel_count(void) { return kernel_count(); }
const char *wd_kernel_name(int id) { return (id >= 0 && id < kernel_count()) ? kernel_info(id).name : nullptr; }

int wd_kernel_for(const wd_handle *h, int nrhs) {
    if (!h || nrhs < 1) return WD_EINVAL;
    if (h->kernel_opt >= 0) return (int)h->kernel_opt;
    return auto_kernel(h, nrhs);
}

int wd_kernel_in_use(const wd_handle *h) { return wd_kernel_for(h, 1); }

long wd_launch_count(const wd_handle *h) { return h ? h->launches : 0; }

int wd_set_option(wd_handle *h, int option, long value) {
    if (!h) return WD_EINVAL;
    h->config_epoch++;  // a captured GMRES cycle has the kernel choice, variant, chunking and link storage baked in
    switch (option) {
    case WD_OPT_VARIANT:
        if (value != 0 && value != 1) return fail(h, WD_EINVAL, "WD_OPT_VARIANT: 0 (fused) or 1 (unfused)");
        h->variant = value;
        return WD_OK;
    case WD_OPT_KERNEL:
        if (value < -1 || value >= kernel_count()) return fail(h, WD_EINVAL, "WD_OPT_KERNEL: id out of range");
        if (value >= 0 && kernel_info((int)value).rhs_block != h->rhs_block)
            return fail(h, WD_EINVAL, std::string("WD_OPT_KERNEL: ") + kernel_info((int)value).name + " is written for WD_OPT_RHS_BLOCK = " + std::to_string(kernel_info((int)value).rhs_block));
        if (value >= 0 && !geometry_fits(h, kernel_info((int)value)))
            return fail(h, WD_EINVAL, std::string("WD_OPT_KERNEL: ") + kernel_info((int)value).name + " does not fit this handle (its tile does not divide the lattice)");
        h->kernel_opt = value;
        return WD_OK;
    case WD_OPT_TCHUNK:
        if (value < 0 || (value > 0 && h->n[0] % value != 0)) return fail(h, WD_EINVAL, "WD_OPT_TCHUNK: must divide T");
        h->tchunk_opt = value;
        return WD_OK;
    case WD_OPT_ZGROUP:
        if (value < 0) return fail(h, WD_EINVAL, "WD_OPT_ZGROUP: must be >= 0");
        h->zgroup_opt = value;
        return WD_OK;
    case WD_OPT_DEVICE_PACK:
        h->device_pack = value ? 1 : 0;
        return WD_OK;
    case WD_OPT_HOST_PIPELINE:
        h->host_pipeline = value ? 1 : 0;
        return WD_OK;
    case WD_OPT_GMRES_GRAPH:
        h->gmres_graph = value ? 1 : 0;
        return WD_OK;
    case WD_OPT_F32_KERNEL:
        if (value != 0 && value != 1) return fail(h, WD_EINVAL, "WD_OPT_F32_KERNEL: 0 (automatic) or 1 (one-thread-per-site kernels)");
        h->f32_kernel = value;
        return WD_OK;
    case WD_OPT_RHS_BLOCK: {
        if (value != 1 && value != 4) return fail(h, WD_EINVAL, "WD_OPT_RHS_BLOCK: 1 (plain layout, default) or 4 (blocked)");
        if (value == 4) {
            bool fits = false;
            for (int id = 0; id < kernel_count(); id++) fits = fits || (kernel_info(id).rhs_block == 4 && geometry_fits(h, kernel_info(id)));
            if (!fits) return fail(h, WD_EINVAL, "WD_OPT_RHS_BLOCK = 4: the 2x4x8 tile of the blocked kernel does not divide this lattice");
            if (h->dd) return fail(h, WD_EINVAL, "WD_OPT_RHS_BLOCK = 4: not available on a decomposed handle (wd_create_local)");
        }
        if (value != h->rhs_block) h->kernel_opt = -1;  // a kernel chosen by hand belongs to the other layout
        h->rhs_block = value;
        return WD_OK;
    }
    case WD_OPT_GAUGE_ROWS: {
        if (value != 2 && value != 3) return fail(h, WD_EINVAL, "WD_OPT_GAUGE_ROWS: 3 (all nine entries, default) or 2 (two-row storage)");
        DeviceGuard guard(h->device);
        h->gauge_rows = value;
        return refresh_two_row_copy(h);
    }
    default:
        return fail(h, WD_EINVAL, "wd_set_option: unknown option");
    }
}

int wd_get_option(const wd_handle *h, int option, long *value) {
    if (!h || !value) return WD_EINVAL;
    switch (option) {
    case WD_OPT_VARIANT: *value = h->variant; return WD_OK;
    case WD_OPT_KERNEL: *value = h->kernel_opt; return WD_OK;
    case WD_OPT_TCHUNK: *value = h->tchunk_opt; return WD_OK;
    case WD_OPT_ZGROUP: *value = h->zgroup_opt; return WD_OK;
    case WD_OPT_DEVICE_PACK: *value = h->device_pack; return WD_OK;
    case WD_OPT_HOST_PIPELINE: *value = h->host_pipeline; return WD_OK;
    case WD_OPT_GMRES_GRAPH: *value = h->gmres_graph; return WD_OK;
    case WD_OPT_GAUGE_ROWS: *value = h->gauge_rows; return WD_OK;
    case WD_OPT_F32_KERNEL: *value = h->f32_kernel; return WD_OK;
    case WD_OPT_RHS_BLOCK: *value = h->rhs_block; return WD_OK;
    default: return WD_EINVAL;
    }
}

// ---- apply ------------------------------------------------------------------------------------------
}  // extern "C"

int wd::fill_params(wd_handle *h, KParams &p, const KernelInfo &k) {
    p.U = h->dU;
    p.U2 = (h->gauge_rows == 2) ? h->dU2 : nullptr;
    p.S = h->dS;
    p.V = h->V;
    p.Vs = h->Vs;
    for (int a = 0; a < 4; a++) p.n[a] = h->n[a];
    p.stride[3] = 1;
    p.stride[2] = h->n[3];
    p.stride[1] = h->n[3] * h->n[2];
    p.stride[0] = h->n[3] * h->n[2] * h->n[1];
    p.mass = h->m0 + 4.0;
    p.ntx = p.nty = p.ntz = p.ntc = p.gz = p.tchunk = 1;
    p.opt_tchunk = (int)h->tchunk_opt;
    p.opt_zgroup = (int)h->zgroup_opt;
    p.tc_begin = p.tc_count = 0;
    p.sched = h->dsched;
    p.nsm = h->nsm;
    p.device = h->device;
    p.maps = h->maps;
    p.open_mask = dd_open_mask(h);
    p.esize = 16;
    p.gauge_rows = (h->gauge_rows == 2 && h->dU2) ? 2 : 3;
    if (k.bx) {
        p.ntx = h->n[3] / k.bx;
        p.nty = h->n[2] / k.by;
        p.ntz = h->n[1] / k.bz;
        long tchunk = h->tchunk_opt;
        if (tchunk == 0) {  // automatic: the largest divisor of T that is <= 16 and a multiple of BT
            tchunk = k.bt;
            for (int c = k.bt; c <= 16 && c <= h->n[0]; c += k.bt)
                if (h->n[0] % c == 0) tchunk = c;
        }
        if (tchunk % k.bt != 0 || h->n[0] % tchunk != 0) return fail(h, WD_EINVAL, "WD_OPT_TCHUNK incompatible with the kernel's T tile");
        p.tchunk = (int)tchunk;
        p.ntc = h->n[0] / p.tchunk;
        long gz = h->zgroup_opt;
        if (gz == 0) gz = p.ntz;  // automatic: one group (whole Z range)
        if (gz > p.ntz || p.ntz % gz != 0) return fail(h, WD_EINVAL, "WD_OPT_ZGROUP must divide the number of Z tiles");
        p.gz = (int)gz;
    }
    return WD_OK;
}

// The TMA kernels expect the two work-queue words to be zero at launch; the last CTA of every launch re-arms them.
// After a failed launch (or a stream change with work pending, see wd_set_stream) they are zeroed explicitly.
int wd::launch_op(wd_handle *h, const KernelInfo &k, const KParams &p, int self) {
    if (h->sched_dirty) {
        WD_CUDA(h, cudaMemsetAsync(h->dsched, 0, 2 * sizeof(unsigned int), h->stream));
        h->sched_dirty = false;
    }
    const cudaError_t e = k.launch(p, self, h->stream);
    if (e != cudaSuccess) {
        h->sched_dirty = true;
        map_cache_clear(h->maps);
        return fail(h, (e == cudaErrorMemoryAllocation) ? WD_ENOMEM : WD_ECUDA, std::string("kernel launch (") + k.name + "): " + cudaGetErrorString(e));
    }
    h->launches++;
    return WD_OK;
}

extern "C" {

int wd_apply(wd_handle *h, void *dev_out, const void *dev_in, int nrhs) {
    WD_ENTER(h);
    if (!dev_out || !dev_in || nrhs < 1) return fail(h, WD_EINVAL, "wd_apply: null pointer or nrhs < 1");
    if (misaligned(dev_out) || misaligned(dev_in)) return fail(h, WD_EINVAL, "wd_apply: spinor buffers must be 16-byte aligned");
    const size_t bytes = wd_spinor_bytes(h, nrhs);
    const char *o = (const char *)dev_out, *i = (const char *)dev_in;
    if (o < i + bytes && i < o + bytes) return fail(h, WD_EINVAL, "wd_apply: out overlaps in");
    if (!h->has_gauge) return fail(h, WD_ESTATE, "wd_apply: no gauge field loaded");
    if (h->csw != 0.0 && !h->has_clover)
        return fail(h, WD_ESTATE, "wd_apply: csw != 0 but no self-coupling field (wd_load_clover / wd_build_clover)");
    const int kid = wd_kernel_for(h, nrhs);
    const KernelInfo &k = kernel_info(kid);
    if (k.rhs_block != h->rhs_block) return fail(h, WD_ESTATE, "wd_apply: no kernel for this spinor layout on this lattice");
    if (h->rhs_block > 1 && h->variant != 0) return fail(h, WD_ESTATE, "wd_apply: the unfused variant reads the plain layout (WD_OPT_RHS_BLOCK = 1)");
    KParams p;
    int rc = fill_params(h, p, k);
    if (rc) return rc;
    const int self = h->has_clover ? SELF_CLOVER : SELF_MASS;
    const size_t per = (size_t)h->Vs * kSpinorComps;
    p.nrhs = 1;
    if (k.multi_rhs && h->variant == 0) {  // a8: one launch, links and S shared by the right-hand sides
        p.psi = (const double2 *)dev_in;
        p.out = (double2 *)dev_out;
        p.nrhs = nrhs;
        return launch_op(h, k, p, self);
    }
    for (int r = 0; r < nrhs; r++) {
        p.psi = (const double2 *)dev_in + r * per;
        p.out = (double2 *)dev_out + r * per;
        if (h->variant == 0) {
            rc = launch_op(h, k, p, self);
            if (rc) return rc;
        } else {
            rc = launch_op(h, k, p, SELF_NONE);
            if (rc) return rc;
            WD_CUDA(h, launch_selfcoupling(p, self, h->stream));
            h->launches++;
        }
    }
    return WD_OK;
}

// Pipelined host-to-host application (TMA kernels, fused variant): the lattice is cut into C chunks along T; chunk
// k is computed as soon as chunks k-1, k, k+1 of the input are on the device and in device layout, and is
// repacked and copied back while the next chunks are computed.  Upload (s_up), compute (the handle's stream) and
// download (s_dn) overlap, so a PCIe-bound application costs about max(H2D, D2H) instead of H2D + D2H.
static int apply_host_pipelined(wd_handle *h, double *host_out, const double *host_in, int nrhs, int C) {
    const int T = h->n[0], tcs = T / C;               // slices per chunk
    const long long Vc = h->V / T * tcs;              // sites per chunk (a T range is a contiguous site range)
    const size_t per = (size_t)h->V * kSpinorComps, cbytes = (size_t)Vc * kSpinorComps * sizeof(double2);
    if (!h->pipe_ready) {
        WD_CUDA(h, cudaStreamCreateWithFlags(&h->s_up, cudaStreamNonBlocking));
        WD_CUDA(h, cudaStreamCreateWithFlags(&h->s_dn, cudaStreamNonBlocking));
        for (int k = 0; k < kMaxPipeChunks; k++) {
            WD_CUDA(h, cudaEventCreateWithFlags(&h->ev_up[k], cudaEventDisableTiming));
            WD_CUDA(h, cudaEventCreateWithFlags(&h->ev_cmp[k], cudaEventDisableTiming));
        }
        WD_CUDA(h, cudaEventCreateWithFlags(&h->ev_misc[0], cudaEventDisableTiming));
        WD_CUDA(h, cudaEventCreateWithFlags(&h->ev_misc[1], cudaEventDisableTiming));
        h->pipe_ready = true;
    }
    // canonical-layout staging on the device: rings of kStageRing chunks (stream order makes a slot's next use wait for
    // its previous one: upload and transpose of a chunk are both on s_up, transpose and download both on s_dn)
    const int kStageRing = 4;
    int rc0 = ensure_dstage(h, (size_t)kStageRing * cbytes);
    if (rc0) return rc0;
    if (h->dstage_out_bytes < (size_t)kStageRing * cbytes) {
        if (h->dstage_out) cudaFree(h->dstage_out);
        h->dstage_out = nullptr;
        h->dstage_out_bytes = 0;
        WD_CUDA(h, cudaMalloc((void **)&h->dstage_out, (size_t)kStageRing * cbytes));
        h->dstage_out_bytes = (size_t)kStageRing * cbytes;
    }
    const size_t celems = (size_t)Vc * kSpinorComps;  // elements per chunk in canonical layout
    long long nup = 0, ndn = 0;                       // chunks uploaded / downloaded so far (ring positions)
    const KernelInfo &kinfo = kernel_info(wd_kernel_in_use(h));
    KParams p;
    const long saved_tchunk = h->tchunk_opt;
    h->tchunk_opt = tcs;
    int rc = fill_params(h, p, kinfo);
    h->tchunk_opt = saved_tchunk;
    if (rc) return rc;
    p.psi = h->work_in;
    p.out = h->work_out;
    p.nrhs = 1;
    p.tc_count = 1;
    const int self = h->has_clover ? SELF_CLOVER : SELF_MASS;
    // everything issued so far on the handle's stream comes first
    WD_CUDA(h, cudaEventRecord(h->ev_misc[0], h->stream));
    WD_CUDA(h, cudaStreamWaitEvent(h->s_up, h->ev_misc[0], 0));
    WD_CUDA(h, cudaStreamWaitEvent(h->s_dn, h->ev_misc[0], 0));
    for (int r = 0; r < nrhs; r++) {
        const double2 *src = (const double2 *)host_in + r * per;
        double2 *dst = (double2 *)host_out + r * per;
        if (r > 0) {  // the previous right-hand side must be out of work_in (compute) and work_out (repack)
            WD_CUDA(h, cudaStreamWaitEvent(h->s_up, h->ev_cmp[C - 1], 0));
            WD_CUDA(h, cudaStreamWaitEvent(h->stream, h->ev_misc[1], 0));
        }
        for (int i = 0; i < C; i++) {  // upload order: last chunk first (chunk 0 needs slice T-1), then 0, 1, ...
            const int k = (i == 0) ? C - 1 : i - 1;
            const long long s0 = (long long)k * Vc;
            double2 *stage = h->dstage + (size_t)(nup++ % kStageRing) * celems;
            WD_CUDA(h, cudaMemcpyAsync(stage, src + s0 * kSpinorComps, cbytes, cudaMemcpyHostToDevice, h->s_up));
            WD_CUDA(h, launch_aos_to_soa(h->work_in + s0, stage, Vc, h->Vs, kSpinorComps, h->s_up));
            WD_CUDA(h, cudaEventRecord(h->ev_up[k], h->s_up));
            h->launches++;
        }
        for (int k = 0; k < C; k++) {
            WD_CUDA(h, cudaStreamWaitEvent(h->stream, h->ev_up[(k + C - 1) % C], 0));
            WD_CUDA(h, cudaStreamWaitEvent(h->stream, h->ev_up[k], 0));
            WD_CUDA(h, cudaStreamWaitEvent(h->stream, h->ev_up[(k + 1) % C], 0));
            p.tc_begin = k;
            rc = launch_op(h, kinfo, p, self);
            if (rc) return rc;
            WD_CUDA(h, cudaEventRecord(h->ev_cmp[k], h->stream));
            const long long s0 = (long long)k * Vc;
            WD_CUDA(h, cudaStreamWaitEvent(h->s_dn, h->ev_cmp[k], 0));
            double2 *stage = h->dstage_out + (size_t)(ndn++ % kStageRing) * celems;
            WD_CUDA(h, launch_soa_to_aos(stage, h->work_out + s0, Vc, h->Vs, kSpinorComps, h->s_dn));
            h->launches++;
            if (k == C - 1) WD_CUDA(h, cudaEventRecord(h->ev_misc[1], h->s_dn));
            WD_CUDA(h, cudaMemcpyAsync(dst + s0 * kSpinorComps, stage, cbytes, cudaMemcpyDeviceToHost, h->s_dn));
        }
    }
    WD_CUDA(h, cudaStreamSynchronize(h->s_dn));
    WD_CUDA(h, cudaStreamSynchronize(h->s_up));
    WD_CUDA(h, cudaStreamSynchronize(h->stream));
    return WD_OK;
}

int wd_apply_host(wd_handle *h, double *host_out, const double *host_in, int nrhs) {
    WD_ENTER(h);
    if (!host_out || !host_in || nrhs < 1) return fail(h, WD_EINVAL, "wd_apply_host: null pointer or nrhs < 1");
    WD_PLAIN_ONLY(h, "wd_apply_host");
    if (!h->has_gauge) return fail(h, WD_ESTATE, "wd_apply_host: no gauge field loaded");
    if (h->csw != 0.0 && !h->has_clover)
        return fail(h, WD_ESTATE, "wd_apply_host: csw != 0 but no self-coupling field (wd_load_clover / wd_build_clover)");
    const size_t per = (size_t)h->V * kSpinorComps, bytes = per * sizeof(double2);
    const size_t dbytes = wd_spinor_bytes(h, 1);
    if (!h->work_in) WD_CUDA(h, cudaMalloc((void **)&h->work_in, dbytes));
    if (!h->work_out) WD_CUDA(h, cudaMalloc((void **)&h->work_out, dbytes));
    // pipelined path (WD_OPT_HOST_PIPELINE, default on): a TMA kernel, fused variant, and T splits into 4..32 equal chunks
    const KernelInfo &kinfo = kernel_info(wd_kernel_in_use(h));
    int C = 0;
    if (kinfo.multi_rhs && h->variant == 0 && h->host_pipeline) {
        for (int c = kMaxPipeChunks; c >= 4 && !C; c--)
            if (h->n[0] % c == 0) C = c;
    }
    if (C) return apply_host_pipelined(h, host_out, host_in, nrhs, C);
    int rc = ensure_dstage(h, bytes);  // the serial path stages a whole right-hand side
    if (rc) return rc;
    for (int r = 0; r < nrhs; r++) {
        WD_CUDA(h, cudaMemcpyAsync(h->dstage, (const double2 *)host_in + r * per, bytes, cudaMemcpyHostToDevice, h->stream));
        WD_CUDA(h, launch_aos_to_soa(h->work_in, h->dstage, h->V, h->Vs, kSpinorComps, h->stream));
        h->launches++;
        rc = wd_apply(h, h->work_out, h->work_in, 1);
        if (rc) return rc;
        WD_CUDA(h, launch_soa_to_aos(h->dstage, h->work_out, h->V, h->Vs, kSpinorComps, h->stream));
        h->launches++;
        WD_CUDA(h, cudaMemcpyAsync((double2 *)host_out + r * per, h->dstage, bytes, cudaMemcpyDeviceToHost, h->stream));
    }
    WD_CUDA(h, cudaStreamSynchronize(h->stream));
    return WD_OK;
}

}  // extern "C"
