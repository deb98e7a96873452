// wd_tma.cu — the Blackwell-native fused Wilson-clover kernel: TMA-staged, warp-specialised,
// marching along T.
//
// out(x) = S(x) psi(x) - 1/2 sum_mu [ (1-gamma_mu) U_mu(x) psi(x+mu) + (1+gamma_mu) U_mu(x-mu)^H psi(x-mu) ]
// (eq. 1.13), steps a1-a7 of SURVEY.md §8(a) in one pass.
//
// Why this shape (round-1 ncu captures of the LDG kernels; summary in DESIGN.md section 5): the one-thread-per-site LDG kernels are latency-bound — the
// bytes in flight per SM are (resident warps) x (registers a thread can spare), and with 140-180
// registers per thread only 8-11 warps fit.  Here the bytes in flight are decoupled from registers:
//   * a persistent CTA (one per SM) owns a BZ x BY x BX tile of sites and marches it along T;
//   * ONE producer thread streams everything the tile needs — own links, the x-mu face links, S,
//     psi and its six spatial faces — into ~222 KB of shared memory with cp.async.bulk.tensor
//     (5-D tensor maps over the SoA fields), each object guarded by a full/empty mbarrier pair;
//   * N = BZ*BY*BX compute threads (one per site) read operands from shared memory only
//     (conflict-free LDS.128 on the SoA boxes), so they never wait on DRAM directly;
//   * each object's buffer is refilled for slice t+1 as soon as slice t has consumed it: at any
//     time all of shared memory except the object being consumed is either landing or waiting,
//     i.e. ~150-200 KB in flight per SM (Little: 6.5 TB/s x ~1 us / 148 SMs = 45 KB needed).
// T direction: psi(t-1) and psi(t+1) are never fetched.  The backward hop of slice t uses the
// half-spinor (1+gamma_T) psi(t-1) carried in registers from the previous step; the forward hop
// of slice t-1 is added when psi(t) arrives, just before out(t-1) is stored (U_T(t-1) is the
// "T object").  So per site and step HBM supplies psi 192 + U 576 + S 576 B and takes 192 B: the
// algorithmic 1536 B, plus face re-reads that hit L2 (neighbouring tiles march concurrently).
// Neighbour indexing and the periodic wrap (a1) are box coordinates computed by the producer.
#include <cstdio>
#include <cstdlib>
#include <new>

#include "wd_tma_plan.cuh"

namespace wd {

// ---------------------------------------------------------------- tensor-map encoder (host)
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

cudaError_t encode_field_map(CUtensorMap *map, const void *base, const int n[4], long long Vs, int ncomp, int bx,
                             int by, int bz, int bc, int esize, int rb) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) return cudaErrorNotSupported;
    const cuuint64_t T = n[0], Z = n[1], Y = n[2], X = n[3];
    const cuuint64_t dims[5] = {2 * X * rb, Y, Z, T, (cuuint64_t)ncomp};
    const cuuint64_t es = (cuuint64_t)esize * rb;  // bytes per site: one complex element, 16 (FP64) or 8 (FP32), times rb
    const cuuint64_t strides[4] = {X * es, X * Y * es, X * Y * Z * es, (cuuint64_t)Vs * es};  // bytes, dims 1..4
    const cuuint32_t box[5] = {(cuuint32_t)(2 * bx * rb), (cuuint32_t)by, (cuuint32_t)bz, 1u, (cuuint32_t)bc};
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    const CUtensorMapL2promotion promo = (bx * es >= 256)   ? CU_TENSOR_MAP_L2_PROMOTION_L2_256B
                                         : (bx * es >= 128) ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B
                                                            : CU_TENSOR_MAP_L2_PROMOTION_NONE;
    const CUresult r = fn(map, (esize == 8) ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, const_cast<void *>(base), dims, strides, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, promo,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return (r == CUDA_SUCCESS) ? cudaSuccess : cudaErrorInvalidValue;
}

MapCache *map_cache_new() { return new (std::nothrow) MapCache(); }
void map_cache_delete(MapCache *c) { delete c; }
void map_cache_clear(MapCache *c) {
    if (c) c->clear();
}

using namespace gen1;

// ---------------------------------------------------------------- the kernel
// OPEN = false: a periodic lattice — the open-boundary predicates fold away (they cost 9 % more instructions)
template <class P, bool OPEN>
__global__ void __launch_bounds__(P::NTHREADS, P::CTAS_PER_SM) k_tma(const __grid_constant__ TmaMaps maps, const TmaParams prm) {
    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t sbase = smem_u32(smem);
    constexpr int OB_SB = P::OB_SB, OB_ITEM0 = P::OB_ITEM0, OB_COUNT = P::OB_COUNT;
    const uint32_t bar_full = sbase + P::OFF_BAR, bar_empty = bar_full + OB_COUNT * 8;
    const int tid = threadIdx.x;
    typedef typename P::C C;
    typedef R<C> Real;
    constexpr int BZ = P::BZ, BY = P::BY, BX = P::BX, N = P::N;
    constexpr bool CLOVER = (P::SELF == SELF_CLOVER);
    const Real half = (Real)0.5, mass = (Real)prm.mass;

    if (tid == 0) {
        if (sbase & 127u) __trap();  // TMA destinations need 128-byte alignment
        for (int k = 0; k < OB_COUNT; k++) {
            mbar_init(bar_full + 8 * k, 1);        // the producer's arrive(.expect_tx)
            mbar_init(bar_empty + 8 * k, P::NW);   // one arrive per compute warp
        }
        mbar_fence_init();
    }
    __syncthreads();

    const int T = prm.n[0], Z = prm.n[1], Y = prm.n[2], X = prm.n[3];

    if (tid >= N) {
        // ======================= producer: one thread issues every TMA (wd_tma_plan.cuh) =======================
        if (tid == N) producer<P, false>(maps, prm, smem, sbase, bar_full, bar_empty);
        return;
    }
    // ======================= consumers: one thread per site of the tile =======================
    const int lane = tid & 31;
    const int lx = tid % BX, ly = (tid / BX) % BY, lz = tid / (BX * BY);
    constexpr uint32_t E = P::E, NS = N * E;
    const uint32_t own = tid * E;
    // operand addresses (bytes from the start of shared memory): interior or face storage
    const uint32_t fz = (ly * BX + lx) * E, fy = (lz * BX + lx) * E;
    // X faces: XW sites per (z, y) row; the neighbour column is the last one of the low face, the first of the high face
    const uint32_t fxl = ((lz * BY + ly) * P::XW + (P::XW - 1)) * E, fxh = ((lz * BY + ly) * P::XW) * E;
    const bool zf_in = lz < BZ - 1, zb_in = lz > 0, yf_in = ly < BY - 1, yb_in = ly > 0, xf_in = lx < BX - 1, xb_in = lx > 0;
    const uint32_t z_pf = zf_in ? P::OFF_C + own + P::FZ * E : P::OFF_ZHI + fz, z_pf_s = zf_in ? NS : P::FZ * E;
    const uint32_t z_pb = zb_in ? P::OFF_C + own - P::FZ * E : P::OFF_ZLO + fz, z_b_s = zb_in ? NS : P::FZ * E;
    const uint32_t z_ub = zb_in ? P::OFF_Z + own - P::FZ * E : P::OFF_ZUF + fz;
    const uint32_t y_pf = yf_in ? P::OFF_C + own + BX * E : P::OFF_YHI + fy, y_pf_s = yf_in ? NS : P::FY * E;
    const uint32_t y_pb = yb_in ? P::OFF_C + own - BX * E : P::OFF_YLO + fy, y_b_s = yb_in ? NS : P::FY * E;
    const uint32_t y_ub = yb_in ? P::OFF_Y + own - BX * E : P::OFF_YUF + fy;
    const uint32_t x_pf = xf_in ? P::OFF_C + own + E : P::OFF_XHI + fxh, x_pf_s = xf_in ? NS : P::FX * E;
    const uint32_t x_pb = xb_in ? P::OFF_C + own - E : P::OFF_XLO + fxl, x_b_s = xb_in ? NS : P::FX * E;
    const uint32_t x_ub = xb_in ? P::OFF_X + own - E : P::OFF_XUF + fxl;

    auto release = [&](int ob) {
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8 * ob);
    };

    const long long V = prm.Vs;  // component stride
    const long long strideT = (long long)Z * Y * X;
    uint32_t nC = 0, nT = 0, nF = 0;  // fills consumed so far
#ifdef WD_EXPERIMENTS
    int ntrace = 0;
#endif
    C hprev[6];                      // rows 0,1 of (1 + gamma_T) psi(t-1)
    C outp[12];                      // out(t-1) still missing its forward-T hop

    const volatile int *mail = reinterpret_cast<const volatile int *>(smem + P::OFF_MAIL);
    for (uint32_t seq = 0;; seq++) {
        const uint32_t slot = P::COMPACT ? 0 : (seq & 1), mpar = P::COMPACT ? (seq & 1) : ((seq >> 1) & 1);
        mbar_wait(bar_full + 8 * (OB_ITEM0 + slot), mpar);
        const int item = mail[slot];
        release(OB_ITEM0 + slot);
        if (item < 0) break;
        const Item it = decode_item<P>(prm, item);
        const long long site0 = ((long long)(it.z0 + lz) * Y + (it.y0 + ly)) * X + (it.x0 + lx);
        C *__restrict__ out = reinterpret_cast<C *>(prm.out) + (long long)it.rhs0 * 12 * V;
        // open boundaries of a domain-decomposed sub-lattice: hops that would cross them are left out
        const int open = OPEN ? prm.open_mask : 0;
        const bool zf_on = !((open & 2) && it.z0 + lz == Z - 1), zb_on = !((open & 2) && it.z0 + lz == 0);
        const bool yf_on = !((open & 4) && it.y0 + ly == Y - 1), yb_on = !((open & 4) && it.y0 + ly == 0);
        const bool xf_on = !((open & 8) && it.x0 + lx == X - 1), xb_on = !((open & 8) && it.x0 + lx == 0);
        int t = (it.t0 == 0) ? T - 1 : it.t0 - 1;
        {   // prologue: seed the carried half-spinor from psi(t0-1)
            C p[12];
            mbar_wait(bar_full + 8 * OB_C, nC & 1);
#pragma unroll
            for (int c = 0; c < 12; c++) p[c] = lds<C>(smem, P::OFF_C + own + c * NS);
            project<0, +1>(hprev, p);
            if ((open & 1) && it.t0 == 0) {
#pragma unroll
                for (int c = 0; c < 6; c++) hprev[c] = mk<C>(0, 0);
            }
            release(OB_C);
            nC++;
        }
        for (int j = 1; j <= prm.tchunk + 1; j++) {
            const int tprev = t;
            t = (t + 1 == T) ? 0 : t + 1;
            C p[12], acc[12];
            {   // T phase: finish out(t-1) with its forward hop, start out(t) with its backward hop
                C u[9];
                mbar_wait(bar_full + 8 * OB_T, nT & 1);
                mbar_wait(bar_full + 8 * OB_C, nC & 1);
#ifdef WD_EXPERIMENTS
                if (prm.trace && tid == 0 && ntrace < kTraceLen) {
                    unsigned long long now;
                    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(now));
                    prm.trace[(size_t)blockIdx.x * kTraceLen + ntrace++] = now;
                }
#endif
                load_link<P::UC, C>(u, smem, P::OFF_T + own, NS);
#pragma unroll
                for (int c = 0; c < 12; c++) p[c] = lds<C>(smem, P::OFF_C + own + c * NS);
                if (j > 1) {  // out(t-1) = outp - 1/2 (1 - gamma_T) U_T(t-1) psi(t)
                    C hf[6], gf[6], o[12];
                    project<0, -1>(hf, p);
                    su3_mul<false>(gf, u, hf);
                    reconstruct_axpy<0, -1>(o, outp, ((open & 1) && tprev == T - 1) ? (Real)0 : -half, gf);
                    const long long ip = (long long)tprev * strideT + site0;
#pragma unroll
                    for (int c = 0; c < 12; c++) __stcs(out + (long long)c * V + ip, o[c]);
                }
                if (j == prm.tchunk + 1) {  // epilogue step: nothing else to do for slice t
                    release(OB_T);
                    release(OB_C);
                    nT++;
                    nC++;
                    break;
                }
                C g[6];
                su3_mul<true>(g, u, hprev);  // U_T(t-1)^H (1 + gamma_T) psi(t-1)
                reconstruct_set<0, +1>(acc, g);
                project<0, +1>(hprev, p);
                release(OB_T);
                nT++;
            }
            const uint32_t pf = nF & 1;
            mbar_wait(bar_full + 8 * OB_Z, pf);
            hop_pair_smem<1, P::UC, C>(acc, smem, P::OFF_Z + own, NS, z_pf, z_pf_s, z_ub, z_b_s, z_pb, z_b_s, zf_on, zb_on);
            release(OB_Z);
            mbar_wait(bar_full + 8 * OB_Y, pf);
            hop_pair_smem<2, P::UC, C>(acc, smem, P::OFF_Y + own, NS, y_pf, y_pf_s, y_ub, y_b_s, y_pb, y_b_s, yf_on, yb_on);
            release(OB_Y);
            mbar_wait(bar_full + 8 * OB_X, pf);
            hop_pair_smem<3, P::UC, C>(acc, smem, P::OFF_X + own, NS, x_pf, x_pf_s, x_ub, x_b_s, x_pb, x_b_s, xf_on, xb_on);
            release(OB_X);
            release(OB_C);
            nC++;
            // self-coupling (a5) and combination (a6); the store waits for the forward-T hop
            if (CLOVER) {
#pragma unroll
                for (int b = 0; b < 2; b++) {
                    const uint32_t so = (b == 0 ? P::OFF_SA : P::OFF_SB) + own;
                    if (!P::COMPACT || b == 0) mbar_wait(bar_full + 8 * (b == 0 ? OB_SA : OB_SB), pf);
                    Real d[6];
                    C a[15], r[6];
#pragma unroll
                    for (int q = 0; q < 3; q++) {
                        const C dd = lds<C>(smem, so + q * NS);
                        d[2 * q] = dd.x;
                        d[2 * q + 1] = dd.y;
                    }
#pragma unroll
                    for (int k = 0; k < 15; k++) a[k] = lds<C>(smem, so + (3 + k) * NS);
                    if (!P::COMPACT || b == 1) release(b == 0 ? OB_SA : OB_SB);
                    herm6_mul(r, d, a, p + 6 * b);
#pragma unroll
                    for (int c = 0; c < 6; c++)
                        outp[6 * b + c] = mk<C>(fma(-half, acc[6 * b + c].x, r[c].x), fma(-half, acc[6 * b + c].y, r[c].y));
                }
            } else if (P::SELF == SELF_MASS) {
#pragma unroll
                for (int c = 0; c < 12; c++)
                    outp[c] = mk<C>(fma(mass, p[c].x, -half * acc[c].x), fma(mass, p[c].y, -half * acc[c].y));
            } else {
#pragma unroll
                for (int c = 0; c < 12; c++) outp[c] = mk<C>(-half * acc[c].x, -half * acc[c].y);
            }
            nF++;
        }
    }
}

// ---------------------------------------------------------------- host side
template <int BZ, int BY, int BX, int SELF> static cudaError_t launch_tma_self(const KParams &p, cudaStream_t st) {
    if (p.esize == 8) {  // FP32 variant: the same kernel on 8-byte elements (pointers of p are float2 fields)
        using P = Plan<BZ, BY, BX, SELF, 9, cf>;
        return p.open_mask ? launch_tma_kernel<P>(k_tma<P, true>, p, st, /*ucomp*/ 9, /*scomp*/ 18, CHUNK_COST_MODEL, /*rb*/ 4) : launch_tma_kernel<P>(k_tma<P, false>, p, st, /*ucomp*/ 9, /*scomp*/ 18, CHUNK_COST_MODEL, /*rb*/ 4);
    }
    if (p.gauge_rows == 2) {  // two-row link storage: boxes of 6 components from the compressed gauge array
        using P = Plan<BZ, BY, BX, SELF, 6>;
        KParams q = p;
        q.U = p.U2;
        return q.open_mask ? launch_tma_kernel<P>(k_tma<P, true>, q, st, /*ucomp*/ 6, /*scomp*/ 18, CHUNK_COST_MODEL, /*rb*/ 4) : launch_tma_kernel<P>(k_tma<P, false>, q, st, /*ucomp*/ 6, /*scomp*/ 18, CHUNK_COST_MODEL, /*rb*/ 4);
    }
    using P = Plan<BZ, BY, BX, SELF>;
    return p.open_mask ? launch_tma_kernel<P>(k_tma<P, true>, p, st, /*ucomp*/ 9, /*scomp*/ 18, CHUNK_COST_MODEL, /*rb*/ 4) : launch_tma_kernel<P>(k_tma<P, false>, p, st, /*ucomp*/ 9, /*scomp*/ 18, CHUNK_COST_MODEL, /*rb*/ 4);
}

template <int BZ, int BY, int BX> static cudaError_t launch_tma(const KParams &p, int self, cudaStream_t st) {
    if (self == SELF_CLOVER) return launch_tma_self<BZ, BY, BX, SELF_CLOVER>(p, st);
    if (self == SELF_MASS) return launch_tma_self<BZ, BY, BX, SELF_MASS>(p, st);
    return launch_tma_self<BZ, BY, BX, SELF_NONE>(p, st);
}

cudaError_t launch_tma_2x4x16(const KParams &p, int self, cudaStream_t st) { return launch_tma<2, 4, 16>(p, self, st); }
}  // namespace wd
