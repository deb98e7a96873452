// wd_gmres.cu — restarted GMRES(m) on the device around the operator: Algorithm 1 of the paper
// with M = I, in the paper's order:
//
//     r = b - A x;  beta = ||r||;  v_1 = r / beta                                     (lines 4-6)
//     for j = 1..m:  w = A v_j                                                        (line 9: wd_apply, the hot path)
//                    for i = 1..j:  h_ij = <w, v_i> = v_i^H w;  w = w - h_ij v_i      (lines 10-12, modified Gram-Schmidt)
//                    h_{j+1,j} = ||w||;  v_{j+1} = w / h_{j+1,j}                       (lines 14-15)
//     y = argmin || beta e_1 - H y ||;  x = x + V y                                   (lines 18-20)
//
// Termination as DDalphaAMG's (R17, R18): ||b - A x|| < tol ||b - A x_0|| tested on
// the true residual at the top of the restart loop, or max_cycles; |h_{j+1,j}| < tol/10 ends the Arnoldi loop.
//
// Vectors are device spinors in DEVICE layout ([12][Vs], the padding between components is never touched).
// The BLAS-1 work is fused so that every pass over memory does as much as the sequential dependence of modified
// Gram-Schmidt allows:  [w -= h_{i-1,j} v_{i-1}  and  h_ij = <w, v_i>]  is ONE kernel (3 reads + 1 write instead of
// 2 + 3 reads and 1 write), the last subtraction is fused with the norm, the solution update reads all basis
// vectors in one pass.  Every scalar (h_ij, beta, 1/h, y, the breakdown flag) lives in device memory and is
// produced by the last block of the kernel that reduces it (fixed summation order: results are deterministic),
// so a whole restart cycle is a fixed sequence of launches without host synchronisation: it is captured once
// into a CUDA graph and replayed (the consumer of cfg 3's "100 back-to-back applications", SURVEY.md:399).
#include <cmath>
#include <cstddef>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "wd_handle.h"
#include "wd_math.cuh"

using namespace wd;

namespace {
constexpr int kMaxM = 64;
constexpr int kThreads = 256;

struct Scalars {          // device-resident scalars of the iteration
    double2 H[(kMaxM + 1) * kMaxM];  // H[i + (m+1) * j]
    double2 y[kMaxM];
    double beta, inv;     // ||r||, and the reciprocal the next scaling uses (1/beta or 1/h_{j+1,j})
    double lsq_resid;     // |g_{kdim+1}|: the recurrence residual of the cycle
    int active, kdim;     // Arnoldi still running; Krylov dimension of this cycle
    int kdim_done;        // Krylov dimension of the cycle that was completed last (kdim is re-armed for the next one)
    unsigned int ticket;  // last-block detection of the reductions (zero between kernels)
};
}  // namespace

struct wd_gmres_state {
    int m;
    double2 *basis;       // (m + 2) device spinors: v_0 .. v_m, w
    int m32;
    float2 *basis32;      // wd_gmres_mixed: (m + 2) single-precision device spinors v_0 .. v_m, w
    double2 *r64;         // wd_gmres_mixed: the FP64 residual b - A x
    Scalars *sc;          // device
    double2 *partials;    // per-block partial sums of the reductions
    int nbx;              // blocks per component
    cudaGraphExec_t graph;
    const void *gx, *gb;  // what the captured cycle was built for
    int gm;
    long gepoch;          // h->config_epoch at capture: options, fields and FP32 copies the cycle has baked in
    bool gmixed;          // the captured cycle is wd_gmres_mixed's
    double gtol;
    cudaStream_t gstream;
    long graph_launches;  // kernel launches inside one captured cycle
    int last_m, last_kdim;
    std::vector<double2> hostH;
};

namespace {

__device__ __forceinline__ double2 block_reduce(double2 v, double2 *sh) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        v.x += __shfl_xor_sync(0xffffffffu, v.x, o);
        v.y += __shfl_xor_sync(0xffffffffu, v.y, o);
    }
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) sh[w] = v;
    __syncthreads();
    v = (threadIdx.x < kThreads / 32) ? sh[threadIdx.x] : make_double2(0.0, 0.0);
    if (w == 0) {
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) {
            v.x += __shfl_xor_sync(0xffffffffu, v.x, o);
            v.y += __shfl_xor_sync(0xffffffffu, v.y, o);
        }
    }
    return v;  // valid in thread 0
}

// Grid-wide sum in a fixed order: every block leaves its partial, the last block to finish adds them up.
// Returns true in thread 0 of that last block, with the total in *total.
__device__ __forceinline__ bool grid_reduce(double2 mine, double2 *partials, unsigned int *ticket, double2 *total) {
    __shared__ double2 sh[kThreads / 32];
    __shared__ bool last;
    const unsigned int nblk = gridDim.x * gridDim.y, blk = blockIdx.y * gridDim.x + blockIdx.x;
    const double2 b = block_reduce(mine, sh);
    if (threadIdx.x == 0) {
        partials[blk] = b;
        __threadfence();
        last = (atomicAdd(ticket, 1u) == nblk - 1);
    }
    __syncthreads();
    if (!last) return false;
    __threadfence();
    double2 s = make_double2(0.0, 0.0);
    for (unsigned int k = threadIdx.x; k < nblk; k += kThreads) {
        const double2 p = partials[k];
        s.x += p.x;
        s.y += p.y;
    }
    s = block_reduce(s, sh);
    if (threadIdx.x == 0) {
        *total = s;
        *ticket = 0;
        return true;
    }
    return false;
}

enum { OP_DOT = 0, OP_AXPY_DOT, OP_AXPY_NORM, OP_RESID_NORM };

// One fused pass (see the header): the vectors are [12][Vs], blockIdx.y is the component.
//   OP_DOT        : h_out = <w, vn>
//   OP_AXPY_DOT   : w -= h_in * vp;  h_out = <w, vn>
//   OP_AXPY_NORM  : w -= h_in * vp;  h_out = ||w|| (real), inv = 1 / h_out, breakdown rule
//   OP_RESID_NORM : w = bvec - w;    beta = ||w||, inv = 1 / beta; starts a cycle (active = 1, kdim = m)
// CV = element type of the vectors: double2, or float2 (wd_gmres_mixed: single-precision Krylov vectors; every product and
// sum is still formed in double, only the stored vector is rounded)
template <class CV> __device__ __forceinline__ double2 ldv(const CV *p, long long i) {
    const CV v = p[i];
    return make_double2((double)v.x, (double)v.y);
}
template <class CV> __device__ __forceinline__ void stv(CV *p, long long i, double2 v) { p[i] = mk<CV>((R<CV>)v.x, (R<CV>)v.y); }
// A thread moves 16 bytes per access: one double2, or two consecutive float2 (i even; the component base is a multiple of
// 16 elements).  n = elements that exist (the last access of an odd-length component holds one).
template <class CV> struct Epa { static constexpr int n = 16 / (int)sizeof(CV); };
template <class CV> __device__ __forceinline__ void ldn(const CV *p, long long i, int n, double2 *x) {
    if (Epa<CV>::n == 2) {
        if (n == 2) {
            const float4 v = *reinterpret_cast<const float4 *>(p + i);
            x[0] = make_double2((double)v.x, (double)v.y);
            x[1] = make_double2((double)v.z, (double)v.w);
        } else {
            x[0] = ldv(p, i);
            x[1] = make_double2(0.0, 0.0);
        }
    } else {
        x[0] = ldv(p, i);
    }
}
template <class CV> __device__ __forceinline__ void stn(CV *p, long long i, int n, const double2 *x) {
    if (Epa<CV>::n == 2 && n == 2) *reinterpret_cast<float4 *>(p + i) = make_float4((float)x[0].x, (float)x[0].y, (float)x[1].x, (float)x[1].y);
    else stv(p, i, x[0]);
}

template <int OP, class CV>
__global__ void __launch_bounds__(kThreads) k_fused(CV *__restrict__ w, const CV *__restrict__ vp,
                                                    const CV *__restrict__ vn, long long V, long long Vs, Scalars *sc,
                                                    int h_in, int h_out, int j, int m, double tol10) {
    if (OP != OP_RESID_NORM && !sc->active) return;
    const long long base = (long long)blockIdx.y * Vs;
    double2 h = make_double2(0.0, 0.0);
    if (OP == OP_AXPY_DOT || OP == OP_AXPY_NORM) h = sc->H[h_in];
    double2 acc = make_double2(0.0, 0.0);
    constexpr int E = Epa<CV>::n;
    const long long nacc = (V + E - 1) / E;
    for (long long a = (long long)blockIdx.x * kThreads + threadIdx.x; a < nacc; a += (long long)gridDim.x * kThreads) {
        const long long i = a * E;
        const int n = (V - i < E) ? (int)(V - i) : E;
        double2 x[E], p[E], q[E];
        ldn(w, base + i, n, x);
        if (OP == OP_AXPY_DOT || OP == OP_AXPY_NORM) {
            ldn(vp, base + i, n, p);
#pragma unroll
            for (int e = 0; e < E; e++) {
                x[e].x = fma(-h.x, p[e].x, fma(h.y, p[e].y, x[e].x));
                x[e].y = fma(-h.x, p[e].y, fma(-h.y, p[e].x, x[e].y));
                if (sizeof(CV) == sizeof(float2)) x[e] = make_double2((double)(float)x[e].x, (double)(float)x[e].y);  // the inner product sees the vector as stored
            }
            stn(w, base + i, n, x);
        } else if (OP == OP_RESID_NORM) {
            ldn(vp, base + i, n, p);
#pragma unroll
            for (int e = 0; e < E; e++) x[e] = make_double2(p[e].x - x[e].x, p[e].y - x[e].y);
            stn(w, base + i, n, x);
        }
        if (OP == OP_DOT || OP == OP_AXPY_DOT) {  // conj(vn) * x
            ldn(vn, base + i, n, q);
#pragma unroll
            for (int e = 0; e < E; e++) {
                acc.x = fma(q[e].x, x[e].x, fma(q[e].y, x[e].y, acc.x));
                acc.y = fma(q[e].x, x[e].y, fma(-q[e].y, x[e].x, acc.y));
            }
        } else {
#pragma unroll
            for (int e = 0; e < E; e++) acc.x = fma(x[e].x, x[e].x, fma(x[e].y, x[e].y, acc.x));
        }
    }
    double2 total;
    if (!grid_reduce(acc, reinterpret_cast<double2 *>(sc + 1), &sc->ticket, &total)) return;
    if (OP == OP_DOT || OP == OP_AXPY_DOT) {
        sc->H[h_out] = total;
    } else if (OP == OP_AXPY_NORM) {
        const double hn = sqrt(total.x);
        sc->H[h_out] = make_double2(hn, 0.0);
        sc->inv = (hn > 0.0) ? 1.0 / hn : 0.0;
        if (hn < tol10) {  // near breakdown: the Krylov dimension of this cycle is j + 1
            sc->active = 0;
            sc->kdim = j + 1;
        }
    } else {
        const double beta = sqrt(total.x);
        sc->beta = beta;
        sc->inv = (beta > 0.0) ? 1.0 / beta : 0.0;
        sc->active = 1;
        sc->kdim = m;
    }
}

// dst = inv * src (v_1 = r / beta, v_{j+1} = w / h_{j+1,j}); `always`: also when the Arnoldi loop has ended
template <class CD, class CS>
__global__ void __launch_bounds__(kThreads) k_scale(CD *__restrict__ dst, const CS *__restrict__ src, long long V,
                                                    long long Vs, const Scalars *sc, int always) {
    if (!always && !sc->active) return;
    const double s = sc->inv;
    const long long base = (long long)blockIdx.y * Vs;
    constexpr int E = Epa<CD>::n;  // accesses sized by the destination
    const long long nacc = (V + E - 1) / E;
    for (long long a = (long long)blockIdx.x * kThreads + threadIdx.x; a < nacc; a += (long long)gridDim.x * kThreads) {
        const long long i = a * E;
        const int n = (V - i < E) ? (int)(V - i) : E;
        double2 x[E];
#pragma unroll
        for (int e = 0; e < E; e++) x[e] = (e < n) ? ldv(src, base + i + e) : make_double2(0.0, 0.0);
#pragma unroll
        for (int e = 0; e < E; e++) x[e] = make_double2(s * x[e].x, s * x[e].y);
        stn(dst, base + i, n, x);
    }
}

// y = argmin || beta e_1 - H y ||_2 over the kdim columns of this cycle: Givens QR of the (kdim+1) x kdim Hessenberg
// matrix, one thread (kdim <= 64).  Rotation [[c, s], [-conj(s), c]], c real, zeroes the sub-diagonal entry.
__global__ void k_lsq(Scalars *sc, int m) {
    if (threadIdx.x || blockIdx.x) return;
    const int kd = sc->kdim, ld = m + 1;
    sc->kdim_done = kd;
    double2 g[kMaxM + 1];
    double2 *H = sc->H;
    for (int k = 0; k <= kd; k++) g[k] = make_double2(0.0, 0.0);
    g[0].x = sc->beta;
    for (int k = 0; k < kd; k++) {
        const double2 a = H[k + ld * k];
        const double b = H[k + 1 + ld * k].x;
        const double na = hypot(a.x, a.y), r = hypot(na, b);
        double c = 1.0;
        double2 s = make_double2(0.0, 0.0);
        if (r > 0.0) {
            if (na > 0.0) {
                c = na / r;
                s = make_double2(b * a.x / (na * r), b * a.y / (na * r));
            } else {
                c = 0.0;
                s = make_double2(1.0, 0.0);
            }
        }
        for (int col = k; col < kd; col++) {  // rows k, k+1 of the remaining columns (and of column k itself)
            const double2 p = H[k + ld * col], q = H[k + 1 + ld * col];
            H[k + ld * col] = make_double2(c * p.x + s.x * q.x - s.y * q.y, c * p.y + s.x * q.y + s.y * q.x);
            H[k + 1 + ld * col] = make_double2(-(s.x * p.x + s.y * p.y) + c * q.x, -(s.x * p.y - s.y * p.x) + c * q.y);
        }
        const double2 p = g[k];
        g[k] = make_double2(c * p.x, c * p.y);
        g[k + 1] = make_double2(-(s.x * p.x + s.y * p.y), -(s.x * p.y - s.y * p.x));
    }
    sc->lsq_resid = hypot(g[kd].x, g[kd].y);
    for (int k = kd - 1; k >= 0; k--) {  // back substitution R y = g
        double2 t = g[k];
        for (int col = k + 1; col < kd; col++) {
            const double2 rr = H[k + ld * col], yy = sc->y[col];
            t.x -= rr.x * yy.x - rr.y * yy.y;
            t.y -= rr.x * yy.y + rr.y * yy.x;
        }
        const double2 d = H[k + ld * k];
        const double dd = d.x * d.x + d.y * d.y;
        sc->y[k] = (dd > 0.0) ? make_double2((t.x * d.x + t.y * d.y) / dd, (t.y * d.x - t.x * d.y) / dd) : make_double2(0.0, 0.0);
    }
}

// x += sum_i y_i v_i over the kdim basis vectors of this cycle, one pass (line 19)
template <class CV>
__global__ void __launch_bounds__(kThreads) k_update(double2 *__restrict__ x, const CV *__restrict__ basis, long long V,
                                                     long long Vs, long long vec_stride, const Scalars *sc) {
    const int kd = sc->kdim;
    const long long base = (long long)blockIdx.y * Vs;
    constexpr int E = Epa<CV>::n;
    const long long nacc = (V + E - 1) / E;
    for (long long a = (long long)blockIdx.x * kThreads + threadIdx.x; a < nacc; a += (long long)gridDim.x * kThreads) {
        const long long i = a * E;
        const int n = (V - i < E) ? (int)(V - i) : E;
        double2 s[E], v[E];
#pragma unroll
        for (int e = 0; e < E; e++) s[e] = (e < n) ? x[base + i + e] : make_double2(0.0, 0.0);
        for (int k = 0; k < kd; k++) {
            const double2 yk = sc->y[k];
            ldn(basis, (long long)k * vec_stride + base + i, n, v);
#pragma unroll
            for (int e = 0; e < E; e++) {
                s[e].x = fma(yk.x, v[e].x, fma(-yk.y, v[e].y, s[e].x));
                s[e].y = fma(yk.x, v[e].y, fma(yk.y, v[e].x, s[e].y));
            }
        }
#pragma unroll
        for (int e = 0; e < E; e++)
            if (e < n) x[base + i + e] = s[e];
    }
}

// Hessenberg matrix of the cycle as the Arnoldi process produced it (before k_lsq rotates it in place)
__global__ void k_copy_h(double2 *dst, const Scalars *sc, int n) {
    for (int k = threadIdx.x; k < n; k += blockDim.x) dst[k] = sc->H[k];
}

// the state and the device scalars; then the Krylov vectors of the precision asked for
int ensure_workspace(wd_handle *h, int m, bool mixed) {
    wd_gmres_state *g = h->gmres;
    const size_t vec = (size_t)h->Vs * kSpinorComps * sizeof(double2);
    if (g) {
        if (!mixed && g->m < m) {
            if (g->graph) cudaGraphExecDestroy(g->graph);
            g->graph = nullptr;
            if (g->basis) cudaFree(g->basis);
            g->basis = nullptr;
            g->m = 0;
            WD_CUDA(h, cudaMalloc((void **)&g->basis, (size_t)(m + 2) * vec));
            g->m = m;
        }
        if (mixed && g->m32 < m) {
            if (g->graph) cudaGraphExecDestroy(g->graph);
            g->graph = nullptr;
            if (g->basis32) cudaFree(g->basis32);
            g->basis32 = nullptr;
            g->m32 = 0;
            WD_CUDA(h, cudaMalloc((void **)&g->basis32, (size_t)(m + 2) * vec / 2));
            g->m32 = m;
        }
        if (mixed && !g->r64) WD_CUDA(h, cudaMalloc((void **)&g->r64, vec));
        return WD_OK;
    }
    g = new (std::nothrow) wd_gmres_state();
    if (!g) return fail(h, WD_ENOMEM, "wd_gmres: out of host memory");
    g->m = g->m32 = 0;
    g->basis = nullptr;
    g->basis32 = nullptr;
    g->r64 = nullptr;
    g->sc = nullptr;
    g->graph = nullptr;
    g->gx = g->gb = nullptr;
    g->gepoch = -1;
    g->gmixed = false;
    g->graph_launches = 0;
    g->last_m = g->last_kdim = 0;
    long long nbx = (h->V + kThreads * 8 - 1) / (kThreads * 8);  // ~8 elements per thread, at most ~8 blocks per SM
    const long long cap = (long long)h->nsm * 8 / 12 + 1;
    if (nbx > cap) nbx = cap;
    if (nbx < 1) nbx = 1;
    g->nbx = (int)nbx;
    // the scalars, followed by the per-block partial sums and room for a copy of H; the state is published only once
    // they exist (a handle whose state had no scalars would hand the kernels a null pointer on the next call)
    const size_t extra = (size_t)g->nbx * 12 * sizeof(double2) + (size_t)(kMaxM + 1) * kMaxM * sizeof(double2);
    cudaError_t e = cudaMalloc((void **)&g->sc, sizeof(Scalars) + extra);
    if (e == cudaSuccess) e = cudaMemsetAsync(g->sc, 0, sizeof(Scalars) + extra, h->stream);
    if (e != cudaSuccess) {
        if (g->sc) cudaFree(g->sc);
        delete g;
        WD_CUDA(h, e);
    }
    h->gmres = g;
    return ensure_workspace(h, m, mixed);
}

// Issues the launches of the algorithm on the handle's stream and counts them.  CV = double2: wd_gmres.  CV = float2:
// wd_gmres_mixed — Krylov vectors, operator applications and orthogonalisation in single precision, the residual
// b - A x, the solution x and every scalar in double.
template <class CV> struct Cycle {
    static constexpr bool MIXED = sizeof(CV) == sizeof(float2);
    wd_handle *h;
    wd_gmres_state *g;
    int m;
    double tol10;
    long launches = 0;
    CV *base() const {
        if constexpr (MIXED) return g->basis32;
        else return g->basis;
    }
    CV *vec(int k) const { return base() + (size_t)k * h->Vs * kSpinorComps; }
    CV *w() const { return vec(m + 1); }
    double2 *r() const {  // the FP64 residual vector: w itself, or its own buffer when w is single precision
        if constexpr (MIXED) return g->r64;
        else return w();
    }
    dim3 grid() const { return dim3((unsigned)g->nbx, 12); }
    template <int OP, class T> int fused(T *wv, const T *vp, const T *vn, int h_in, int h_out, int j) {
        k_fused<OP, T><<<grid(), kThreads, 0, h->stream>>>(wv, vp, vn, h->V, h->Vs, g->sc, h_in, h_out, j, m, tol10);
        WD_CUDA(h, cudaGetLastError());
        launches++;
        return WD_OK;
    }
    template <class T> int apply(T *out, const T *in) {
        const long before = h->launches;
        int rc;
        if constexpr (sizeof(T) == sizeof(float2)) rc = wd_apply_f32(h, out, in, 1);
        else rc = wd_apply(h, out, in, 1);
        launches += h->launches - before;
        h->launches = before;  // the caller adds `launches` once per executed cycle (graph replays included)
        return rc;
    }
    // r = b - A x;  beta = ||r||   (always FP64)
    int residual(const double2 *x, const double2 *b) {
        int rc = apply(r(), x);
        if (rc) return rc;
        return fused<OP_RESID_NORM, double2>(r(), b, nullptr, 0, 0, 0);
    }
    // lines 6-20 of Algorithm 1, then line 4-5 for the new x
    int body(double2 *x, const double2 *b) {
        const int ld = m + 1;
        int rc;
        k_scale<CV, double2><<<grid(), kThreads, 0, h->stream>>>(vec(0), r(), h->V, h->Vs, g->sc, 1);  // v_1 = r / beta
        WD_CUDA(h, cudaGetLastError());
        launches++;
        WD_CUDA(h, cudaMemsetAsync(g->sc->H, 0, sizeof(double2) * (size_t)ld * m, h->stream));
        for (int j = 0; j < m; j++) {
            if ((rc = apply(w(), (const CV *)vec(j)))) return rc;                                        // w = A v_j
            if ((rc = fused<OP_DOT, CV>(w(), nullptr, vec(0), 0, 0 + ld * j, j))) return rc;            // h_1j
            for (int i = 1; i <= j; i++)                                                                // w -= h_{i-1,j} v_{i-1}; h_ij
                if ((rc = fused<OP_AXPY_DOT, CV>(w(), vec(i - 1), vec(i), (i - 1) + ld * j, i + ld * j, j))) return rc;
            if ((rc = fused<OP_AXPY_NORM, CV>(w(), vec(j), nullptr, j + ld * j, (j + 1) + ld * j, j))) return rc;
            k_scale<CV, CV><<<grid(), kThreads, 0, h->stream>>>(vec(j + 1), w(), h->V, h->Vs, g->sc, 0);  // v_{j+1}
            WD_CUDA(h, cudaGetLastError());
            launches++;
        }
        double2 *Hcopy = reinterpret_cast<double2 *>(g->sc + 1) + (size_t)g->nbx * 12;
        k_copy_h<<<1, 256, 0, h->stream>>>(Hcopy, g->sc, ld * m);
        k_lsq<<<1, 32, 0, h->stream>>>(g->sc, m);
        k_update<CV><<<grid(), kThreads, 0, h->stream>>>(x, base(), h->V, h->Vs, h->Vs * kSpinorComps, g->sc);
        WD_CUDA(h, cudaGetLastError());
        launches += 3;
        return residual(x, b);
    }
};

}  // namespace

void wd::gmres_free(wd_handle *h) {
    wd_gmres_state *g = h->gmres;
    if (!g) return;
    if (g->graph) cudaGraphExecDestroy(g->graph);
    if (g->basis) cudaFree(g->basis);
    if (g->basis32) cudaFree(g->basis32);
    if (g->r64) cudaFree(g->r64);
    if (g->sc) cudaFree(g->sc);
    delete g;
    h->gmres = nullptr;
}

namespace {

// The restart loop of wd_gmres (CV = double2) and wd_gmres_mixed (CV = float2): argument checks, work space, line 4 for
// x_0, then cycles — the first one launch by launch (all caches warm), the second captured into a CUDA graph that the
// later ones replay (WD_OPT_GMRES_GRAPH, non-default stream) — with one host synchronisation per cycle to read ||b - A x||.
template <class CV>
int gmres_driver(wd_handle *h, const char *name, void *dev_x, const void *dev_b, int m, int max_cycles, double tol, int *cycles_done,
                 double *host_resid) {
    constexpr bool MIXED = sizeof(CV) == sizeof(float2);
    const std::string nm(name);
    if (!dev_x || !dev_b || m < 1 || m > kMaxM || max_cycles < 0 || !(tol > 0.0))
        return fail(h, WD_EINVAL, nm + ": null pointer, m outside 1..64, max_cycles < 0 or tol <= 0");
    if (((size_t)dev_x | (size_t)dev_b) & 15) return fail(h, WD_EINVAL, nm + ": spinor buffers must be 16-byte aligned");
    if (dev_x == dev_b) return fail(h, WD_EINVAL, nm + ": x overlaps b");
    if (!h->has_gauge) return fail(h, WD_ESTATE, nm + ": no gauge field loaded");
    if (MIXED && !h->f32) return fail(h, WD_ESTATE, nm + ": call wd_enable_f32 after loading the fields (single-precision copies of U and S)");
    if (MIXED && !f32_current(h)) return fail(h, WD_ESTATE, nm + ": the FP64 links or S changed after wd_enable_f32; call wd_enable_f32 again");
    int rc = ensure_workspace(h, m, MIXED);
    if (rc) return rc;
    wd_gmres_state *g = h->gmres;
    Cycle<CV> cyc{h, g, m, tol / 10.0};
    double2 *x = (double2 *)dev_x;
    const double2 *b = (const double2 *)dev_b;
    struct { double beta, inv, lsq; int active, kdim, kdim_done; unsigned int ticket; } hs;
    auto read_scalars = [&]() -> int {
        WD_CUDA(h, cudaMemcpyAsync(&hs, &g->sc->beta, sizeof(hs), cudaMemcpyDeviceToHost, h->stream));
        WD_CUDA(h, cudaStreamSynchronize(h->stream));
        return WD_OK;
    };
    static_assert(offsetof(Scalars, ticket) - offsetof(Scalars, beta) == 3 * sizeof(double) + 3 * sizeof(int) && sizeof(hs) == 40, "layout of Scalars");
    // lines 4-5 for x_0
    if ((rc = cyc.residual(x, b))) return rc;
    h->launches += cyc.launches;
    if ((rc = read_scalars())) return rc;
    const double r0 = hs.beta;
    if (host_resid) host_resid[0] = r0;
    int k = 0;
    const bool can_graph = (h->stream != nullptr) && h->gmres_graph;
    while (!(hs.beta < tol * r0) && k < max_cycles && hs.beta != 0.0) {
        const bool have_graph = can_graph && g->graph && g->gepoch == h->config_epoch && g->gx == dev_x && g->gb == dev_b && g->gm == m && g->gtol == tol && g->gstream == h->stream && g->gmixed == MIXED;
        if (have_graph) {
            WD_CUDA(h, cudaGraphLaunch(g->graph, h->stream));
            h->launches += g->graph_launches;
        } else if (can_graph && k >= 1) {  // the first cycle ran eagerly (all caches warm): capture the second, replay it
            if (g->graph) cudaGraphExecDestroy(g->graph);
            g->graph = nullptr;
            cudaGraph_t graph = nullptr;
            WD_CUDA(h, cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal));
            cyc.launches = 0;
            rc = cyc.body(x, b);
            const cudaError_t ce = cudaStreamEndCapture(h->stream, &graph);
            if (rc) {
                if (graph) cudaGraphDestroy(graph);
                return rc;
            }
            WD_CUDA(h, ce);
            const cudaError_t ie = cudaGraphInstantiate(&g->graph, graph, 0);
            cudaGraphDestroy(graph);
            WD_CUDA(h, ie);
            g->gx = dev_x, g->gb = dev_b, g->gm = m, g->gtol = tol, g->gstream = h->stream, g->gmixed = MIXED;
            g->gepoch = h->config_epoch;
            g->graph_launches = cyc.launches;
            WD_CUDA(h, cudaGraphLaunch(g->graph, h->stream));
            h->launches += g->graph_launches;
        } else {
            cyc.launches = 0;
            if ((rc = cyc.body(x, b))) return rc;
            h->launches += cyc.launches;
        }
        if ((rc = read_scalars())) return rc;
        k++;
        if (host_resid) host_resid[k] = hs.beta;
    }
    if (cycles_done) *cycles_done = k;
    g->last_m = m;
    g->last_kdim = (k > 0) ? hs.kdim_done : 0;
    return WD_OK;
}

}  // namespace

extern "C" {

int wd_gmres(wd_handle *h, void *dev_x, const void *dev_b, int m, int max_cycles, double tol, int *cycles_done,
             double *host_resid) {
    WD_ENTER(h);
    WD_PLAIN_ONLY(h, "wd_gmres");
    return gmres_driver<double2>(h, "wd_gmres", dev_x, dev_b, m, max_cycles, tol, cycles_done, host_resid);
}

int wd_gmres_mixed(wd_handle *h, void *dev_x, const void *dev_b, int m, int max_cycles, double tol, int *cycles_done,
                   double *host_resid) {
    WD_ENTER(h);
    WD_PLAIN_ONLY(h, "wd_gmres_mixed");
    return gmres_driver<float2>(h, "wd_gmres_mixed", dev_x, dev_b, m, max_cycles, tol, cycles_done, host_resid);
}

int wd_gmres_last_hessenberg(wd_handle *h, double *host_H, int *kdim, double *lsq_resid) {
    WD_ENTER(h);
    wd_gmres_state *g = h->gmres;
    if (!g || g->last_m < 1) return fail(h, WD_ESTATE, "wd_gmres_last_hessenberg: no GMRES cycle has run on this handle");
    const int m = g->last_m;
    if (host_H) {
        const double2 *Hcopy = reinterpret_cast<const double2 *>(g->sc + 1) + (size_t)g->nbx * 12;
        WD_CUDA(h, cudaMemcpyAsync(host_H, Hcopy, sizeof(double2) * (size_t)(m + 1) * m, cudaMemcpyDeviceToHost, h->stream));
    }
    if (lsq_resid) WD_CUDA(h, cudaMemcpyAsync(lsq_resid, &g->sc->lsq_resid, sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    WD_CUDA(h, cudaStreamSynchronize(h->stream));
    if (kdim) *kdim = g->last_kdim;
    return WD_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------------
// wd_inner_product_static — the inner product of lines 10-11 / the norm of lines 5, 14 of Algorithm 1
// for callers that must not allocate (include/wd.h has the contract).  It is k_fused<OP_DOT> with the same grid-wide
// reduction (grid_reduce above: one partial per block, the last block adds them in a fixed order), but the per-block
// partials and the completion counters — which wd_gmres keeps in cudaMalloc'ed memory behind its Scalars — live in a
// fixed array inside the library image.  Nothing below calls cudaMalloc / cudaFree or anything that allocates.
namespace {

constexpr int kStaticSlots = 4096;    // per-block partial sums (16 B each), shared by the right-hand sides of a call
constexpr int kStaticMaxRhs = 64;     // one completion counter per right-hand side
constexpr int kStaticTicketSlots = kStaticMaxRhs * (int)sizeof(unsigned int) / (int)sizeof(double2);  // 16 double2 = 64 counters
constexpr int kStaticMaxDevices = 64;

// 64 KiB + 256 B per GPU that loads libwd.so, for the life of the process.  [0, kStaticSlots): partials;
// the last 256 bytes: the counters.  Shared by every call on the device; holds whatever the last call left.
static __device__ __align__(256) double2 g_static_scratch[kStaticSlots + kStaticTicketSlots];

// g_static_scratch as a host expression is only a shadow the runtime uses to look the symbol up; its DEVICE address, which
// differs from GPU to GPU, is asked for once per device (with that device current) and kept here.
std::mutex g_static_mutex;
double2 *g_static_addr[kStaticMaxDevices];
int g_static_nsm[kStaticMaxDevices];

// result[r] = sum over the 12 components and V sites of conj(a) * b, right-hand side r = blockIdx.z
__global__ void __launch_bounds__(kThreads) k_dot_static(const double2 *__restrict__ a, const double2 *__restrict__ b, long long V,
                                                         long long Vs, double2 *scratch, double2 *__restrict__ result) {
    const long long base = ((long long)blockIdx.z * 12 + blockIdx.y) * Vs;
    double2 acc = make_double2(0.0, 0.0);
    for (long long i = (long long)blockIdx.x * kThreads + threadIdx.x; i < V; i += (long long)gridDim.x * kThreads) {
        const double2 q = a[base + i], x = b[base + i];
        acc.x = fma(q.x, x.x, fma(q.y, x.y, acc.x));
        acc.y = fma(q.x, x.y, fma(-q.y, x.x, acc.y));
    }
    const unsigned int nblk = gridDim.x * gridDim.y;
    unsigned int *tickets = reinterpret_cast<unsigned int *>(scratch + kStaticSlots);
    double2 total;
    if (grid_reduce(acc, scratch + (size_t)blockIdx.z * nblk, tickets + blockIdx.z, &total)) result[blockIdx.z] = total;
}

int static_fail(int code, const std::string &msg) { return fail(nullptr, code, "wd_inner_product_static: " + msg); }

}  // namespace

extern "C" int wd_inner_product_static(const void *dev_a, const void *dev_b, long long V, long long Vs, int nrhs, void *dev_result,
                                       void *cuda_stream) {
    // argument checks first: they need no GPU
    if (!dev_a || !dev_b || !dev_result) return static_fail(WD_EINVAL, "null pointer");
    if (V < 1 || Vs < V || V >= (1LL << 40)) return static_fail(WD_EINVAL, "need 1 <= V <= Vs and V < 2^40");
    if (nrhs < 1) return static_fail(WD_EINVAL, "nrhs < 1");
    if (nrhs > kStaticMaxRhs)
        return static_fail(WD_EINVAL, "nrhs = " + std::to_string(nrhs) + " is beyond the maximum of " + std::to_string(kStaticMaxRhs) +
                                          " right-hand sides per call that the fixed scratch array (" +
                                          std::to_string(sizeof(double2) * (kStaticSlots + kStaticTicketSlots)) +
                                          " bytes, never grown) has counters and partial-sum slots for; split the call");
    if (((size_t)dev_a | (size_t)dev_b | (size_t)dev_result) & 15) return static_fail(WD_EINVAL, "pointers must be 16-byte aligned");
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    int dev = -1;
    WD_CUDA(nullptr, cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return static_fail(WD_EINVAL, "device ordinal beyond " + std::to_string(kStaticMaxDevices - 1));
    double2 *scratch;
    int nsm;
    {  // first call on this device: look the array's device address up (the set-up step the header documents)
        std::lock_guard<std::mutex> lock(g_static_mutex);
        if (!g_static_addr[dev]) {
            double2 *p = nullptr;
            WD_CUDA(nullptr, cudaGetSymbolAddress((void **)&p, g_static_scratch));
            int n = 0;
            WD_CUDA(nullptr, cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev));
            if (!p || n < 1) return static_fail(WD_ECUDA, "no device address for the scratch array");
            g_static_nsm[dev] = n;
            g_static_addr[dev] = p;
        }
        scratch = g_static_addr[dev];
        nsm = g_static_nsm[dev];
    }
    // blocks per component: as wd_gmres (about 8 elements per thread, at most ~8 blocks per SM over the 12 components), and no
    // more than the partial-sum slots allow; nrhs <= 64 leaves at least 5
    long long nbx = (V + kThreads * 8 - 1) / (kThreads * 8);
    const long long cap = (long long)nsm * 8 / 12 + 1, fit = kStaticSlots / (12LL * nrhs);
    if (nbx > cap) nbx = cap;
    if (nbx > fit) nbx = fit;
    if (nbx < 1) nbx = 1;
    // the counters must start at zero; a call that failed half-way may have left them otherwise
    WD_CUDA(nullptr, cudaMemsetAsync(scratch + kStaticSlots, 0, sizeof(double2) * kStaticTicketSlots, stream));
    k_dot_static<<<dim3((unsigned)nbx, 12, (unsigned)nrhs), kThreads, 0, stream>>>((const double2 *)dev_a, (const double2 *)dev_b, V, Vs,
                                                                                  scratch, (double2 *)dev_result);
    WD_CUDA(nullptr, cudaGetLastError());
    return WD_OK;
}
