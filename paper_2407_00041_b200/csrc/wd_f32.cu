// wd_f32.cu — the FP32 variant of the operator (the paper's PRECISION templating):
// the same kernels instantiated on float2 — the TMA-staged T-marching kernel of wd_tma.cu on 8-byte elements where its
// tile divides the lattice, the one-thread-per-site kernels of wd_ldg_kernels.cuh otherwise — on single-precision copies
// of the links and of S that live beside the FP64 fields.  Halves every byte of the path (768 instead of 1536 algorithmic B/site); all
// arithmetic, including the accumulation over the eight hops, is FP32 — the error budget is derived in DESIGN.md
// ("Tolerance of the FP32 variant").  Device layout: the FP64 layout with 8-byte elements, float2 [nrhs][12][Vs].
#include <cstring>
#include <new>

#include "wd_handle.h"
#include "wd_ldg_kernels.cuh"

using namespace wd;

struct wd_f32_state {
    float2 *dU, *dS;
    bool has_clover;
    long fields_epoch;  // h->fields_epoch when the copies were made
};

namespace {

// dst = (float) src or dst = (double) src, element by element over n complex numbers
template <class D, class S> __global__ void __launch_bounds__(256) k_convert(D *__restrict__ dst, const S *__restrict__ src, long long n) {
    for (long long i = (long long)blockIdx.x * 256 + threadIdx.x; i < n; i += (long long)gridDim.x * 256) {
        const S v = src[i];
        dst[i] = mk<D>((R<D>)v.x, (R<D>)v.y);
    }
}

template <class D, class S> cudaError_t convert(D *dst, const S *src, long long n, int nsm, cudaStream_t st) {
    long long blocks = (n + 255) / 256;
    if (blocks > (long long)nsm * 16) blocks = (long long)nsm * 16;
    k_convert<D, S><<<(unsigned)blocks, 256, 0, st>>>(dst, src, n);
    return cudaGetLastError();
}

}  // namespace

bool wd::f32_current(const wd_handle *h) { return h->f32 && h->f32->dU && h->f32->fields_epoch == h->fields_epoch; }

void wd::f32_free(wd_handle *h) {
    if (!h->f32) return;
    if (h->f32->dU) cudaFree(h->f32->dU);
    if (h->f32->dS) cudaFree(h->f32->dS);
    delete h->f32;
    h->f32 = nullptr;
}

extern "C" {

int wd_enable_f32(wd_handle *h) {
    WD_ENTER(h);
    if (!h->has_gauge) return fail(h, WD_ESTATE, "wd_enable_f32: no gauge field loaded");
    if (h->csw != 0.0 && !h->has_clover) return fail(h, WD_ESTATE, "wd_enable_f32: csw != 0 but no self-coupling field");
    if (!h->f32) {
        h->f32 = new (std::nothrow) wd_f32_state();
        if (!h->f32) return fail(h, WD_ENOMEM, "wd_enable_f32: out of host memory");
        h->f32->dU = h->f32->dS = nullptr;
        h->f32->has_clover = false;
    }
    wd_f32_state *f = h->f32;
    h->config_epoch++;
    f->fields_epoch = -1;  // not current until both conversions are enqueued
    if (!f->dU) WD_CUDA(h, cudaMalloc((void **)&f->dU, (size_t)h->Vs * kGaugeComps * sizeof(float2)));
    WD_CUDA(h, convert(f->dU, h->dU, h->Vs * kGaugeComps, h->nsm, h->stream));
    h->launches++;
    f->has_clover = h->has_clover;
    if (h->has_clover) {
        if (!f->dS) WD_CUDA(h, cudaMalloc((void **)&f->dS, (size_t)h->Vs * kCloverSlots * sizeof(float2)));
        WD_CUDA(h, convert(f->dS, h->dS, h->Vs * kCloverSlots, h->nsm, h->stream));
        h->launches++;
    }
    f->fields_epoch = h->fields_epoch;
    return WD_OK;
}

size_t wd_spinor_bytes_f32(const wd_handle *h, int nrhs) {
    if (!h || nrhs < 1) return 0;
    return (size_t)nrhs * (size_t)h->Vs * kSpinorComps * sizeof(float2);
}

int wd_convert_spinor(wd_handle *h, void *dev_dst, const void *dev_src, int nrhs, int to_f32) {
    WD_ENTER(h);
    WD_PLAIN_ONLY(h, "wd_convert_spinor");
    if (!dev_dst || !dev_src || nrhs < 1) return fail(h, WD_EINVAL, "wd_convert_spinor: null pointer or nrhs < 1");
    const long long n = (long long)nrhs * h->Vs * kSpinorComps;
    if (to_f32) WD_CUDA(h, convert((float2 *)dev_dst, (const double2 *)dev_src, n, h->nsm, h->stream));
    else WD_CUDA(h, convert((double2 *)dev_dst, (const float2 *)dev_src, n, h->nsm, h->stream));
    h->launches++;
    return WD_OK;
}

int wd_apply_f32(wd_handle *h, void *dev_out, const void *dev_in, int nrhs) {
    WD_ENTER(h);
    WD_PLAIN_ONLY(h, "wd_apply_f32");
    if (!dev_out || !dev_in || nrhs < 1) return fail(h, WD_EINVAL, "wd_apply_f32: null pointer or nrhs < 1");
    if (((size_t)dev_out | (size_t)dev_in) & 7) return fail(h, WD_EINVAL, "wd_apply_f32: spinor buffers must be 8-byte aligned");
    const size_t bytes = wd_spinor_bytes_f32(h, nrhs);
    const char *o = (const char *)dev_out, *i = (const char *)dev_in;
    if (o < i + bytes && i < o + bytes) return fail(h, WD_EINVAL, "wd_apply_f32: out overlaps in");
    if (!h->f32 || !h->f32->dU) return fail(h, WD_ESTATE, "wd_apply_f32: call wd_enable_f32 after loading the fields");
    if (!f32_current(h))
        return fail(h, WD_ESTATE, "wd_apply_f32: the FP64 links or S changed after wd_enable_f32; call wd_enable_f32 again (the FP32 copies are stale)");
    if (h->csw != 0.0 && !h->f32->has_clover) return fail(h, WD_ESTATE, "wd_apply_f32: no FP32 self-coupling field (wd_enable_f32)");
    const int self = h->f32->has_clover ? SELF_CLOVER : SELF_MASS;
    // geometry: the TMA kernel (the FP64 skeleton on 8-byte elements) where its 2x4x16 tile divides the lattice, else
    // the one-thread-per-site kernels: 1x4x4x16 tiles, or the linear kernel for any extents
    const bool tma = h->f32_kernel != 1 && h->n[1] % 2 == 0 && h->n[2] % 4 == 0 && h->n[3] % 16 == 0;
    const bool tiled = h->n[1] % 4 == 0 && h->n[2] % 4 == 0 && h->n[3] % 16 == 0;
    const KernelInfo *ki = nullptr;
    for (int id = 0; id < kernel_count(); id++)
        if (!strcmp(kernel_info(id).name, tma ? "tma_2x4x16" : tiled ? "tile_1x4x4x16" : "linear256")) ki = &kernel_info(id);
    KParams p;
    int rc = fill_params(h, p, *ki);
    if (rc) return rc;
    if (tma) {  // one launch for all right-hand sides; the field pointers of p are float2 arrays (p.esize = 8)
        p.psi = (const double2 *)dev_in;
        p.out = (double2 *)dev_out;
        p.U = (const double2 *)h->f32->dU;
        p.S = (const double2 *)h->f32->dS;
        p.U2 = nullptr;
        p.gauge_rows = 3;
        p.esize = 8;
        p.nrhs = nrhs;
        return launch_op(h, *ki, p, self);
    }
    const size_t per = (size_t)h->Vs * kSpinorComps;
    for (int r = 0; r < nrhs; r++) {
        const KP<cf> q = make_kp<cf>(p, (const cf *)dev_in + r * per, h->f32->dU, h->f32->dS, (cf *)dev_out + r * per);
        cudaError_t e;
        if (tiled) e = launch_tiled_t<1, 4, 4, 16, cf>(q, self, h->stream);
        else e = launch_linear_t<256, cf>(q, self, h->stream);
        WD_CUDA(h, e);
        h->launches++;
    }
    return WD_OK;
}

}  // extern "C"
