// wd_dd.cu — the operator on a sub-lattice of a domain decomposition: the communication half of
// Algorithm 3 for hyper-rectangular local lattices P_i (eqs. 2.1-2.4).
//
// In a decomposed direction mu the local lattice does not wrap.  What crosses the seam are projected half-spinors,
// 6 complex numbers = 96 B per face site instead of the 192 B of a spinor:
//     lambda_mu(x) = rows 0,1 of (I4 - gamma_mu) psi(x)                 for x on the LOW face  (x_mu = 0),
//                    sent in the NEGATIVE mu direction (Alg. 3 lines 3, 7): the neighbour's sites x - mu need psi(x);
//     chi_mu(x+mu) = rows 0,1 of (I4 + gamma_mu) (x) U_mu(x)^H psi(x)   for x on the HIGH face (x_mu = n_mu - 1),
//                    sent in the POSITIVE mu direction (lines 11, 15): the link multiplication is done by the sender,
//                    so no ghost links are needed anywhere.
// The factor 1/2 of Alg. 3 is applied once, together with the sign, when the result is accumulated (R10).
// One application on a sub-lattice is
//     wd_dd_pack        faces of psi -> send buffers                                    (this file, tiny)
//     [exchange]        the caller moves send buffers into the neighbours' receive buffers (NCCL send/recv, peer
//                       copies, or plain device copies when several sub-lattices live on one device) ...
//     wd_apply          ... while the fused kernel computes everything that needs no neighbour: hops across the open
//                       boundaries are left out (TmaParams::open_mask / KParams::open_mask)
//     wd_dd_exterior    out(x) -= 1/2 (I4 - gamma_mu) (x) U_mu(x) lambda_recv   on the high face  (lines 18-24),
//                       out(x) -= 1/2 (I4 + gamma_mu)-reconstruction of chi_recv on the low face  (lines 26-31).
// Face sites are enumerated in canonical order of the three remaining coordinates (X fastest), which is the same on
// both sides of a seam; buffers are double2 [nrhs][6][F_mu], F_mu = V / n_mu.
#include <new>

#include "wd_handle.h"
#include "wd_math.cuh"

using namespace wd;

struct wd_dd_state {
    int global_dims[4], grid[4], coords[4];
    int open_mask;
};

namespace {

struct FaceGeom {
    long long F;        // face sites
    long long Vs;       // component stride
    int n[4];           // local extents
    long long stride[4];
};

// canonical site index of face site f of direction MU at coordinate c_mu
template <int MU> __device__ __forceinline__ long long face_site(const FaceGeom &g, long long f, int cmu) {
    int c[4];
    long long r = f;
#pragma unroll
    for (int a = 3; a >= 0; a--) {
        if (a == MU) {
            c[a] = cmu;
        } else {
            c[a] = (int)(r % g.n[a]);
            r /= g.n[a];
        }
    }
    return ((long long)(c[0] * g.n[1] + c[1]) * g.n[2] + c[2]) * g.n[3] + c[3];
}

// blockIdx.y = right-hand side, blockIdx.z = 0: low face -> lambda (send_minus), 1: high face -> chi (send_plus)
template <int MU>
__global__ void __launch_bounds__(128) k_dd_pack(const cd *__restrict__ psi, const cd *__restrict__ U, cd *__restrict__ send_minus,
                                                 cd *__restrict__ send_plus, FaceGeom g) {
    const long long f = (long long)blockIdx.x * 128 + threadIdx.x;
    if (f >= g.F) return;
    const bool hi = blockIdx.z == 1;
    const long long i = face_site<MU>(g, f, hi ? g.n[MU] - 1 : 0);
    const cd *__restrict__ p = psi + (long long)blockIdx.y * 12 * g.Vs + i;
    cd q[12], h[6];
#pragma unroll
    for (int c = 0; c < 12; c++) q[c] = __ldg(p + (long long)c * g.Vs);
    cd *__restrict__ dst = (hi ? send_plus : send_minus) + (long long)blockIdx.y * 6 * g.F + f;
    if (!hi) {
        project<MU, -1>(h, q);
#pragma unroll
        for (int c = 0; c < 6; c++) dst[(long long)c * g.F] = h[c];
    } else {
        cd u[9], w[6];
#pragma unroll
        for (int k = 0; k < 9; k++) u[k] = __ldg(U + (long long)(MU * 9 + k) * g.Vs + i);
        project<MU, +1>(h, q);
        su3_mul<true>(w, u, h);
#pragma unroll
        for (int c = 0; c < 6; c++) dst[(long long)c * g.F] = w[c];
    }
}

// HI = true: high face, lambda from the +mu neighbour; HI = false: low face, chi from the -mu neighbour
template <int MU, bool HI>
__global__ void __launch_bounds__(128) k_dd_exterior(cd *__restrict__ out, const cd *__restrict__ U, const cd *__restrict__ recv,
                                                     FaceGeom g) {
    const long long f = (long long)blockIdx.x * 128 + threadIdx.x;
    if (f >= g.F) return;
    const long long i = face_site<MU>(g, f, HI ? g.n[MU] - 1 : 0);
    const cd *__restrict__ r = recv + (long long)blockIdx.y * 6 * g.F + f;
    cd h[6], acc[12];
#pragma unroll
    for (int c = 0; c < 6; c++) h[c] = __ldg(r + (long long)c * g.F);
#pragma unroll
    for (int c = 0; c < 12; c++) acc[c] = make_double2(0.0, 0.0);
    if (HI) {
        cd u[9], w[6];
#pragma unroll
        for (int k = 0; k < 9; k++) u[k] = __ldg(U + (long long)(MU * 9 + k) * g.Vs + i);
        su3_mul<false>(w, u, h);
        reconstruct_add<MU, -1>(acc, w);
    } else {
        reconstruct_add<MU, +1>(acc, h);
    }
    cd *__restrict__ o = out + (long long)blockIdx.y * 12 * g.Vs + i;
#pragma unroll
    for (int c = 0; c < 12; c++) {
        cd v = o[(long long)c * g.Vs];
        v.x = fma(-0.5, acc[c].x, v.x);
        v.y = fma(-0.5, acc[c].y, v.y);
        o[(long long)c * g.Vs] = v;
    }
}

FaceGeom geom(const wd_handle *h, int mu) {
    FaceGeom g;
    g.F = h->V / h->n[mu];
    g.Vs = h->Vs;
    for (int a = 0; a < 4; a++) g.n[a] = h->n[a];
    g.stride[3] = 1;
    g.stride[2] = h->n[3];
    g.stride[1] = (long long)h->n[3] * h->n[2];
    g.stride[0] = (long long)h->n[3] * h->n[2] * h->n[1];
    return g;
}

bool decomposed(const wd_handle *h, int mu) { return h->dd && mu >= 0 && mu < 4 && (h->dd->open_mask >> mu & 1); }

}  // namespace

void wd::dd_free(wd_handle *h) {
    delete h->dd;
    h->dd = nullptr;
}

int wd::dd_open_mask(const wd_handle *h) { return h->dd ? h->dd->open_mask : 0; }

extern "C" {

int wd_create_local(wd_handle **out, const int *global_dims, const int *proc_grid, const int *proc_coords, double m0,
                    double csw) {
    if (!out) return fail(nullptr, WD_EINVAL, "wd_create_local: null handle pointer");
    *out = nullptr;
    if (!global_dims || !proc_grid || !proc_coords) return fail(nullptr, WD_EINVAL, "wd_create_local: null pointer");
    int n[4], mask = 0;
    for (int a = 0; a < 4; a++) {
        if (proc_grid[a] < 1 || global_dims[a] < 1 || global_dims[a] % proc_grid[a] != 0 || proc_coords[a] < 0 ||
            proc_coords[a] >= proc_grid[a])
            return fail(nullptr, WD_EINVAL, "wd_create_local: the process grid must divide the global lattice, coordinates inside the grid");
        n[a] = global_dims[a] / proc_grid[a];
        if (proc_grid[a] > 1) mask |= 1 << a;
    }
    wd_handle *h = nullptr;
    int rc = wd_create(&h, n[0], n[1], n[2], n[3], m0, csw);
    if (rc) return rc;
    h->dd = new (std::nothrow) wd_dd_state();
    if (!h->dd) {
        wd_destroy(h);
        return fail(nullptr, WD_ENOMEM, "wd_create_local: out of host memory");
    }
    for (int a = 0; a < 4; a++) h->dd->global_dims[a] = global_dims[a], h->dd->grid[a] = proc_grid[a], h->dd->coords[a] = proc_coords[a];
    h->dd->open_mask = mask;
    *out = h;
    return WD_OK;
}

int wd_dd_open_mask(const wd_handle *h) { return h ? dd_open_mask(h) : 0; }

long long wd_dd_face_sites(const wd_handle *h, int mu) { return (h && decomposed(h, mu)) ? h->V / h->n[mu] : 0; }

size_t wd_dd_face_bytes(const wd_handle *h, int mu, int nrhs) {
    return (h && decomposed(h, mu) && nrhs >= 1) ? (size_t)nrhs * 6 * (size_t)(h->V / h->n[mu]) * sizeof(double2) : 0;
}

int wd_dd_pack(wd_handle *h, const void *dev_in, int nrhs, int mu, void *dev_send_minus, void *dev_send_plus) {
    WD_ENTER(h);
    WD_PLAIN_ONLY(h, "wd_dd_pack");
    if (!dev_in || !dev_send_minus || !dev_send_plus || nrhs < 1) return fail(h, WD_EINVAL, "wd_dd_pack: null pointer or nrhs < 1");
    if (!decomposed(h, mu)) return fail(h, WD_EINVAL, "wd_dd_pack: direction is not decomposed on this handle");
    if (!h->has_gauge) return fail(h, WD_ESTATE, "wd_dd_pack: no gauge field loaded");
    const FaceGeom g = geom(h, mu);
    const dim3 grid((unsigned)((g.F + 127) / 128), (unsigned)nrhs, 2);
    const cd *psi = (const cd *)dev_in;
    cd *sm = (cd *)dev_send_minus, *sp = (cd *)dev_send_plus;
    switch (mu) {
    case 0: k_dd_pack<0><<<grid, 128, 0, h->stream>>>(psi, h->dU, sm, sp, g); break;
    case 1: k_dd_pack<1><<<grid, 128, 0, h->stream>>>(psi, h->dU, sm, sp, g); break;
    case 2: k_dd_pack<2><<<grid, 128, 0, h->stream>>>(psi, h->dU, sm, sp, g); break;
    default: k_dd_pack<3><<<grid, 128, 0, h->stream>>>(psi, h->dU, sm, sp, g); break;
    }
    WD_CUDA(h, cudaGetLastError());
    h->launches++;
    return WD_OK;
}

int wd_dd_exterior(wd_handle *h, void *dev_out, int nrhs, int mu, const void *dev_recv_from_plus, const void *dev_recv_from_minus) {
    WD_ENTER(h);
    WD_PLAIN_ONLY(h, "wd_dd_exterior");
    if (!dev_out || !dev_recv_from_plus || !dev_recv_from_minus || nrhs < 1)
        return fail(h, WD_EINVAL, "wd_dd_exterior: null pointer or nrhs < 1");
    if (!decomposed(h, mu)) return fail(h, WD_EINVAL, "wd_dd_exterior: direction is not decomposed on this handle");
    if (!h->has_gauge) return fail(h, WD_ESTATE, "wd_dd_exterior: no gauge field loaded");
    const FaceGeom g = geom(h, mu);
    const dim3 grid((unsigned)((g.F + 127) / 128), (unsigned)nrhs, 1);
    cd *o = (cd *)dev_out;
    const cd *rp = (const cd *)dev_recv_from_plus, *rm = (const cd *)dev_recv_from_minus;
    // two launches: with n_mu = 1 the high and the low face are the same sites
#define WD_EXT(MU)                                                         \
    k_dd_exterior<MU, true><<<grid, 128, 0, h->stream>>>(o, h->dU, rp, g); \
    k_dd_exterior<MU, false><<<grid, 128, 0, h->stream>>>(o, h->dU, rm, g);
    switch (mu) {
    case 0: WD_EXT(0) break;
    case 1: WD_EXT(1) break;
    case 2: WD_EXT(2) break;
    default: WD_EXT(3) break;
    }
#undef WD_EXT
    WD_CUDA(h, cudaGetLastError());
    h->launches += 2;
    return WD_OK;
}

}  // extern "C"
