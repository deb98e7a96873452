// wd_tmw.cu — the warpgroup-split fused kernel ("tmw_*"): the first-generation TMA kernel of wd_tma.cu with TWO compute
// warpgroups per tile, eight compute warps per SM instead of four.
//
// Why (round 2 measurements): with one warp per SM sub-partition nothing hides the LDS / DFMA / mbarrier latencies of
// the compute threads; the FP32 instance of wd_tma.cu, whose plan fits twice into an SM, gained 27 % from the second
// CTA (profiles/r2_bench_lines.md).  The FP64 plan (227 KB) fits once, and a thread cannot be split over two threads of
// ONE register budget: 288 threads x 255 registers do not exist (round 1: 168 registers, spills).  Blackwell's
// `setmaxnreg` moves the budget instead: the kernel starts 3 warpgroups at 168 registers, the producer warpgroup
// shrinks to 40 and the two compute warpgroups grow to 232 each.
//
// The work of a site is split by DIRECTION, so that no link, no psi neighbour and no S entry is read twice:
//     warpgroup A (threads   0..127, thread = site):  T hops (with the register-carried state of wd_tma.cu), Z hops,
//                                                      S block A (spins 0,1), the combination and all stores;
//     warpgroup B (threads 128..255, thread = site):  X hops, Y hops, S block B (spins 2,3).
// B hands its twelve partial sums per site to A through shared memory once per step.  The hand-over buffer is the
// Y object itself: B reads it last, overwrites it with its result and signals a named barrier; A reads, fences the
// generic-proxy writes against the next TMA fill, and releases the Y buffer to the producer.  Everything else —
// objects, tensor maps, item queue, T marching — is wd_tma.cu's.  The producer's order follows the new release order:
// T, Z, X, psi, S_A, S_B, Y.
#include <cstdio>
#include <cstdlib>

#include "wd_tma_plan.cuh"

namespace wd {
namespace tmw {

using namespace gen1;  // OB_C .. OB_SA, the plan and the producer of the first generation (wd_tma_plan.cuh)
enum { OB_SB = OB_SA + 1, OB_ITEM0, OB_ITEM1, OB_COUNT };

// The first generation's plan (FP64, nine-entry links) with three warpgroups of N threads
template <int BZ_, int BY_, int BX_, int SELF_> struct Plan : gen1::Plan<BZ_, BY_, BX_, SELF_, 9, cd> {
    typedef gen1::Plan<BZ_, BY_, BX_, SELF_, 9, cd> Base;
    static constexpr int NTHREADS = 3 * Base::N;  // warpgroups A, B and the producer's
    static constexpr int CTAS_PER_SM = 1;
    static_assert(Base::N == 128, "a compute warpgroup is 128 threads");
    static_assert(Base::SZ_Y >= 12 * Base::N * Base::E, "the Y object doubles as the hand-over buffer of warpgroup B");
    static_assert(!Base::COMPACT && Base::OB_SB == OB_SB && Base::OB_ITEM0 == OB_ITEM0 && Base::OB_COUNT == OB_COUNT, "barrier layout");
};

// named barrier 1: warpgroup B arrives when its partial sums are in shared memory, warpgroup A waits for them
__device__ __forceinline__ void handover_arrive() { asm volatile("bar.arrive 1, 256;" ::: "memory"); }
__device__ __forceinline__ void handover_wait() { asm volatile("bar.sync 1, 256;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

template <class P, bool OPEN>
__global__ void __launch_bounds__(P::NTHREADS, 1) k_tmw(const __grid_constant__ TmaMaps maps, const TmaParams prm) {
    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t sbase = smem_u32(smem);
    const uint32_t bar_full = sbase + P::OFF_BAR, bar_empty = bar_full + OB_COUNT * 8;
    const int tid = threadIdx.x;
    constexpr int BZ = P::BZ, BY = P::BY, BX = P::BX, N = P::N, NW = P::NW;
    constexpr bool CLOVER = (P::SELF == SELF_CLOVER);

    if (tid == 0) {
        if (sbase & 127u) __trap();
        // consumer warps that release each object: psi and the mailbox both warpgroups; T, Z, S_A and (after the
        // hand-over) Y warpgroup A; X and S_B warpgroup B
        const int rel[OB_COUNT] = {2 * NW, NW, NW, NW, NW, NW, NW, 2 * NW, 2 * NW};
        for (int k = 0; k < OB_COUNT; k++) {
            mbar_init(bar_full + 8 * k, 1);
            mbar_init(bar_empty + 8 * k, rel[k]);
        }
        mbar_fence_init();
    }
    __syncthreads();

    const int T = prm.n[0], Z = prm.n[1], Y = prm.n[2], X = prm.n[3];
    const int wg = tid / N;  // 0: A, 1: B, 2: producer

    if (wg == 2) {
        // ======================= producer warpgroup: one thread issues every TMA =======================
        reg_dec<40>();
        if (tid == 2 * N) producer<P, true>(maps, prm, smem, sbase, bar_full, bar_empty);
        return;
    }
    // ======================= compute warpgroups: thread = site =======================
    reg_inc<232>();
    const int stid = tid - wg * N;
    const int lane = tid & 31;
    const int lx = stid % BX, ly = (stid / BX) % BY, lz = stid / (BX * BY);
    constexpr uint32_t E = P::E, NS = N * E;
    const uint32_t own = stid * E;
    const uint32_t fz = (ly * BX + lx) * E, fy = (lz * BX + lx) * E, fx = (lz * BY + ly) * E;
    const bool zf_in = lz < BZ - 1, zb_in = lz > 0, yf_in = ly < BY - 1, yb_in = ly > 0, xf_in = lx < BX - 1, xb_in = lx > 0;

    auto release = [&](int ob) {
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8 * ob);
    };

    const long long V = prm.Vs;
    const long long strideT = (long long)Z * Y * X;
    const volatile int *mail = reinterpret_cast<const volatile int *>(smem + P::OFF_MAIL);
    uint32_t nC = 0, nT = 0, nF = 0;

    if (wg == 0) {
        // ---------------------------------------------------------------- warpgroup A: T, Z, S_A, combination, stores
        const uint32_t z_pf = zf_in ? P::OFF_C + own + P::FZ * E : P::OFF_ZHI + fz, z_pf_s = zf_in ? NS : P::FZ * E;
        const uint32_t z_pb = zb_in ? P::OFF_C + own - P::FZ * E : P::OFF_ZLO + fz, z_b_s = zb_in ? NS : P::FZ * E;
        const uint32_t z_ub = zb_in ? P::OFF_Z + own - P::FZ * E : P::OFF_ZUF + fz;
        cd hprev[6];   // rows 0,1 of (1 + gamma_T) psi(t-1)
        cd outp[12];   // out(t-1) still missing its forward-T hop
        for (uint32_t seq = 0;; seq++) {
            const uint32_t slot = seq & 1, mpar = (seq >> 1) & 1;
            mbar_wait(bar_full + 8 * (OB_ITEM0 + slot), mpar);
            const int item = mail[slot];
            release(OB_ITEM0 + slot);
            if (item < 0) break;
            const Item it = decode_item<P>(prm, item);
            const long long site0 = ((long long)(it.z0 + lz) * Y + (it.y0 + ly)) * X + (it.x0 + lx);
            cd *__restrict__ out = reinterpret_cast<cd *>(prm.out) + (long long)it.rhs0 * 12 * V;
            const int open = OPEN ? prm.open_mask : 0;
            const bool zf_on = !((open & 2) && it.z0 + lz == Z - 1), zb_on = !((open & 2) && it.z0 + lz == 0);
            int t = (it.t0 == 0) ? T - 1 : it.t0 - 1;
            {   // prologue: seed the carried half-spinor from psi(t0-1)
                cd p[12];
                mbar_wait(bar_full + 8 * OB_C, nC & 1);
#pragma unroll
                for (int c = 0; c < 12; c++) p[c] = lds(smem, P::OFF_C + own + c * NS);
                project<0, +1>(hprev, p);
                if ((open & 1) && it.t0 == 0) {
#pragma unroll
                    for (int c = 0; c < 6; c++) hprev[c] = make_double2(0.0, 0.0);
                }
                release(OB_C);
                nC++;
            }
            for (int j = 1; j <= prm.tchunk + 1; j++) {
                const int tprev = t;
                t = (t + 1 == T) ? 0 : t + 1;
                cd p[12], acc[12];
                {   // T phase: finish out(t-1) with its forward hop, start out(t) with its backward hop
                    cd u[9];
                    mbar_wait(bar_full + 8 * OB_T, nT & 1);
                    mbar_wait(bar_full + 8 * OB_C, nC & 1);
                    load_link<9>(u, smem, P::OFF_T + own, NS);
#pragma unroll
                    for (int c = 0; c < 12; c++) p[c] = lds(smem, P::OFF_C + own + c * NS);
                    if (j > 1) {  // out(t-1) = outp - 1/2 (1 - gamma_T) U_T(t-1) psi(t)
                        cd hf[6], gf[6], o[12];
                        project<0, -1>(hf, p);
                        su3_mul<false>(gf, u, hf);
                        reconstruct_axpy<0, -1>(o, outp, ((open & 1) && tprev == T - 1) ? 0.0 : -0.5, gf);
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
                    cd g[6];
                    su3_mul<true>(g, u, hprev);  // U_T(t-1)^H (1 + gamma_T) psi(t-1)
                    reconstruct_set<0, +1>(acc, g);
                    project<0, +1>(hprev, p);
                    release(OB_T);
                    nT++;
                }
                const uint32_t pf = nF & 1;
                mbar_wait(bar_full + 8 * OB_Z, pf);
                hop_pair_smem<1>(acc, smem, P::OFF_Z + own, NS, z_pf, z_pf_s, z_ub, z_b_s, z_pb, z_b_s, zf_on, zb_on);
                release(OB_Z);
                release(OB_C);  // psi(t) of the own site is in registers (p), the Z neighbours are done
                nC++;
                if (CLOVER) {   // S block A on spins 0,1; spins 2,3 come from warpgroup B
                    mbar_wait(bar_full + 8 * OB_SA, pf);
                    double d[6];
                    cd a[15], r[6];
#pragma unroll
                    for (int q = 0; q < 3; q++) {
                        const cd dd = lds(smem, P::OFF_SA + own + q * NS);
                        d[2 * q] = dd.x;
                        d[2 * q + 1] = dd.y;
                    }
#pragma unroll
                    for (int k = 0; k < 15; k++) a[k] = lds(smem, P::OFF_SA + own + (3 + k) * NS);
                    release(OB_SA);
                    herm6_mul(r, d, a, p);
#pragma unroll
                    for (int c = 0; c < 6; c++) outp[c] = make_double2(fma(-0.5, acc[c].x, r[c].x), fma(-0.5, acc[c].y, r[c].y));
#pragma unroll
                    for (int c = 6; c < 12; c++) outp[c] = make_double2(-0.5 * acc[c].x, -0.5 * acc[c].y);
                } else if (P::SELF == SELF_MASS) {
#pragma unroll
                    for (int c = 0; c < 12; c++)
                        outp[c] = make_double2(fma(prm.mass, p[c].x, -0.5 * acc[c].x), fma(prm.mass, p[c].y, -0.5 * acc[c].y));
                } else {
#pragma unroll
                    for (int c = 0; c < 12; c++) outp[c] = make_double2(-0.5 * acc[c].x, -0.5 * acc[c].y);
                }
                // hand-over: the twelve partial sums of warpgroup B (already scaled) sit where the Y object was
                handover_wait();
#pragma unroll
                for (int c = 0; c < 12; c++) {
                    const cd b = lds(smem, P::OFF_Y + own + c * NS);
                    outp[c].x += b.x;
                    outp[c].y += b.y;
                }
                fence_proxy_async();  // B's generic-proxy writes (ordered before us by the barrier) vs the next TMA fill
                release(OB_Y);
                nF++;
            }
        }
    } else {
        // ---------------------------------------------------------------- warpgroup B: X, Y, S_B
        const uint32_t y_pf = yf_in ? P::OFF_C + own + BX * E : P::OFF_YHI + fy, y_pf_s = yf_in ? NS : P::FY * E;
        const uint32_t y_pb = yb_in ? P::OFF_C + own - BX * E : P::OFF_YLO + fy, y_b_s = yb_in ? NS : P::FY * E;
        const uint32_t y_ub = yb_in ? P::OFF_Y + own - BX * E : P::OFF_YUF + fy;
        const uint32_t x_pf = xf_in ? P::OFF_C + own + E : P::OFF_XHI + fx, x_pf_s = xf_in ? NS : P::FX * E;
        const uint32_t x_pb = xb_in ? P::OFF_C + own - E : P::OFF_XLO + fx, x_b_s = xb_in ? NS : P::FX * E;
        const uint32_t x_ub = xb_in ? P::OFF_X + own - E : P::OFF_XUF + fx;
        for (uint32_t seq = 0;; seq++) {
            const uint32_t slot = seq & 1, mpar = (seq >> 1) & 1;
            mbar_wait(bar_full + 8 * (OB_ITEM0 + slot), mpar);
            const int item = mail[slot];
            release(OB_ITEM0 + slot);
            if (item < 0) break;
            const Item it = decode_item<P>(prm, item);
            const int open = OPEN ? prm.open_mask : 0;
            const bool yf_on = !((open & 4) && it.y0 + ly == Y - 1), yb_on = !((open & 4) && it.y0 + ly == 0);
            const bool xf_on = !((open & 8) && it.x0 + lx == X - 1), xb_on = !((open & 8) && it.x0 + lx == 0);
            // prologue: psi(t0-1) is for warpgroup A only
            mbar_wait(bar_full + 8 * OB_C, nC & 1);
            release(OB_C);
            nC++;
            for (int j = 1; j <= prm.tchunk + 1; j++) {
                mbar_wait(bar_full + 8 * OB_C, nC & 1);
                if (j == prm.tchunk + 1) {  // epilogue step: psi(t) serves warpgroup A's last forward-T hop
                    release(OB_C);
                    nC++;
                    break;
                }
                cd acc[12], q[6];
#pragma unroll
                for (int c = 0; c < 12; c++) acc[c] = make_double2(0.0, 0.0);
                const uint32_t pf = nF & 1;
                mbar_wait(bar_full + 8 * OB_X, pf);
                hop_pair_smem<3>(acc, smem, P::OFF_X + own, NS, x_pf, x_pf_s, x_ub, x_b_s, x_pb, x_b_s, xf_on, xb_on);
                release(OB_X);
                mbar_wait(bar_full + 8 * OB_Y, pf);
                hop_pair_smem<2>(acc, smem, P::OFF_Y + own, NS, y_pf, y_pf_s, y_ub, y_b_s, y_pb, y_b_s, yf_on, yb_on);
                if (CLOVER) {
#pragma unroll
                    for (int c = 0; c < 6; c++) q[c] = lds(smem, P::OFF_C + own + (6 + c) * NS);  // spins 2,3 of psi(t)
                }
                release(OB_C);
                nC++;
#pragma unroll
                for (int c = 0; c < 12; c++) acc[c] = make_double2(-0.5 * acc[c].x, -0.5 * acc[c].y);
                if (CLOVER) {
                    mbar_wait(bar_full + 8 * OB_SB, pf);
                    double d[6];
                    cd a[15], r[6];
#pragma unroll
                    for (int k = 0; k < 3; k++) {
                        const cd dd = lds(smem, P::OFF_SB + own + k * NS);
                        d[2 * k] = dd.x;
                        d[2 * k + 1] = dd.y;
                    }
#pragma unroll
                    for (int k = 0; k < 15; k++) a[k] = lds(smem, P::OFF_SB + own + (3 + k) * NS);
                    release(OB_SB);
                    herm6_mul(r, d, a, q);
#pragma unroll
                    for (int c = 0; c < 6; c++) {
                        acc[6 + c].x += r[c].x;
                        acc[6 + c].y += r[c].y;
                    }
                }
                // every thread of this warpgroup must be done READING the Y object before anyone overwrites it
                asm volatile("bar.sync 2, 128;" ::: "memory");
#pragma unroll
                for (int c = 0; c < 12; c++) *reinterpret_cast<cd *>(smem + P::OFF_Y + own + c * NS) = acc[c];
                __threadfence_block();
                handover_arrive();
                nF++;
            }
        }
    }
}

// ---------------------------------------------------------------- host side
template <int BZ, int BY, int BX, int SELF> static cudaError_t launch_self(const KParams &p, cudaStream_t st) {
    using P = Plan<BZ, BY, BX, SELF>;
    return p.open_mask ? launch_tma_kernel<P>(k_tmw<P, true>, p, st, 9, 18, CHUNK_COST_MODEL, 4)
                       : launch_tma_kernel<P>(k_tmw<P, false>, p, st, 9, 18, CHUNK_COST_MODEL, 4);
}
template <int BZ, int BY, int BX> static cudaError_t launch(const KParams &p, int self, cudaStream_t st) {
    if (self == SELF_CLOVER) return launch_self<BZ, BY, BX, SELF_CLOVER>(p, st);
    if (self == SELF_MASS) return launch_self<BZ, BY, BX, SELF_MASS>(p, st);
    return launch_self<BZ, BY, BX, SELF_NONE>(p, st);
}
}  // namespace tmw

cudaError_t launch_tmw_2x4x16(const KParams &p, int self, cudaStream_t st) { return tmw::launch<2, 4, 16>(p, self, st); }
}  // namespace wd
