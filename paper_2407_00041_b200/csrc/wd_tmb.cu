// wd_tmb.cu — second generation of the TMA-staged fused kernel ("tmb_*"): psi double-buffered, the
// accumulator is the only state a thread carries.
//
// Same operator, same decomposition (persistent CTA per SM, one producer thread, one compute thread per
// site of a 128-site tile marching along T, atomic work queue) as wd_tma.cu.  What changed:
//   * psi(t) sits in one of TWO buffers for the whole of step t, and psi(t+1) lands in the other one
//     during the step: no operand has less than a full step to arrive (in wd_tma.cu psi(t+1) had only the
//     S phases, and consumers spent 23 % of their samples waiting for it, profiles/r1c);
//   * at the end of step t both T hops that involve U_T(t) are done together: the forward hop completes
//     out(t), which is stored at once, and the backward hop of slice t+1 initialises the next accumulator.
//     Nothing but acc[12] lives across phases (wd_tma.cu also carried out(t-1), (1+gamma_T) psi(t-1) and
//     psi(t): 120 more registers), psi of the own site is re-read from shared memory where it is needed;
//   * S psi is folded into the accumulator (out = -1/2 (hops - 2 S psi)), S arrives as four 9-component
//     objects through a ring of four slots that also carries U_T.
// Measured at 64^4 (profiles/r1c): pure Wilson 3.66 -> 2.96 ms; Wilson-clover 4.17 -> 4.36 ms (the ring and
// the 4x4x8 tile cost more than the registers bring), which is why wd_api.cu picks tma_* when there is a
// clover term and tmb_* when there is none.
#include <cstdio>
#include <cstdlib>

#include "wd_tma_common.cuh"
#include "wd_smem_ops.cuh"

namespace wd {
namespace tmb {

// ---------------------------------------------------------------- shared-memory plan
// Objects (each with a full/empty mbarrier pair):
//   C   psi(t) interior [12][N], TWO buffers (fill n in buffer n & 1): psi(t) is read during the whole of
//       step t and psi(t+1) at its end, so the next slice lands while the current one is in use
//   Z   U_Z(t) interior | U_Z face z0-1 | psi faces z0-1, z0+BZ      [9][N] [9][FZ] [12][FZ] [12][FZ]
//   Y   same for Y;  X  same for X
//   R   a ring of four [9][N] slots shared by the five 9-component objects of a step, in this order:
//       S1, S2 (block A of S(t): 3 diagonal pairs + 6 entries | 9 entries), S3, S4 (block B), T = U_T(t)
//       (consumed between the Y and X hops, and at the end of the step)
enum { OB_C = 0, OB_C1, OB_Z, OB_Y, OB_X, OB_R, OB_R1, OB_R2, OB_R3, OB_ITEM0, OB_ITEM1, OB_COUNT };

// KR = slots of the ring (4; 3 lets the 2x4x16 tile fit)
template <int BZ_, int BY_, int BX_, int SELF_, int KR_ = 4> struct Plan {
    static constexpr int BZ = BZ_, BY = BY_, BX = BX_, SELF = SELF_, KR = KR_;
    static constexpr int G = 1;              // right-hand sides per work item
    static constexpr bool BLK = false;       // plain multi-RHS layout only
    static constexpr int RBK = 1;
    static constexpr int N = BZ * BY * BX;   // sites per tile = compute threads
    static constexpr int CTAS_PER_SM = 1;
    static constexpr int XW = 1;             // sites per row of an X-face box (wd_tma.cu: 2 for 8-byte elements)
    static constexpr int NW = N / 32;        // compute warps
    static constexpr int NTHREADS = N + 32;  // + the producer warp
    static constexpr int FZ = BY * BX, FY = BZ * BX, FX = BZ * BY;  // sites per face
    static constexpr uint32_t E = 16;                               // bytes per element
    static constexpr uint32_t SZ_C = 12 * N * E, SZ_U = 9 * N * E;
    static constexpr uint32_t OFF_C = 0;
    static constexpr uint32_t OFF_Z = OFF_C + 2 * SZ_C;
    static constexpr uint32_t OFF_ZUF = OFF_Z + SZ_U, OFF_ZLO = OFF_ZUF + 9 * FZ * E, OFF_ZHI = OFF_ZLO + 12 * FZ * E;
    static constexpr uint32_t SZ_Z = SZ_U + (9 + 24) * FZ * E;
    static constexpr uint32_t OFF_Y = OFF_Z + SZ_Z;
    static constexpr uint32_t OFF_YUF = OFF_Y + SZ_U, OFF_YLO = OFF_YUF + 9 * FY * E, OFF_YHI = OFF_YLO + 12 * FY * E;
    static constexpr uint32_t SZ_Y = SZ_U + (9 + 24) * FY * E;
    static constexpr uint32_t OFF_X = OFF_Y + SZ_Y;
    static constexpr uint32_t OFF_XUF = OFF_X + SZ_U, OFF_XLO = OFF_XUF + 9 * FX * E, OFF_XHI = OFF_XLO + 12 * FX * E;
    static constexpr uint32_t SZ_X = SZ_U + (9 + 24) * FX * E;
    static constexpr uint32_t OFF_R = OFF_X + SZ_X;
    static constexpr uint32_t OFF_BAR = OFF_R + KR * SZ_U;
    static constexpr uint32_t OFF_MAIL = OFF_BAR + 2 * OB_COUNT * 8;  // int[2]: item index per mailbox slot
    static constexpr uint32_t SMEM = OFF_MAIL + 16;
    static constexpr int RING_PER_STEP = (SELF == SELF_CLOVER) ? 5 : 1;  // S1..S4 and T, or T alone
    static_assert(N % 32 == 0 && FZ % 8 == 0 && FY % 8 == 0 && FX % 8 == 0, "tile faces must keep 128-byte alignment");
    static_assert(SMEM <= 232448, "shared-memory plan exceeds 227 KB");
};

// ---------------------------------------------------------------- the producer (one thread)
// A resumable state machine: advance() performs the next load of the fixed sequence if the buffer it
// targets has been released, else returns false.  Sequence per work item:
//   [fetch item] [psi(t0-1)] [U_T(t0-1)] [psi(t0)]  then per step t:  [Z] [Y] [S1] [S2] [S3] [S4] [X] [psi(t+1)] [U_T(t)]
// — the order in which the consumers release the buffers of the previous step.
enum { ST_FETCH = 0, ST_PRO_C, ST_PRO_T, ST_PRO_C2, ST_Z, ST_S1, ST_Y, ST_S2, ST_X, ST_S3, ST_S4, ST_C, ST_T };

template <class P> struct Producer {
    uint32_t nC, nR, nF, seq;  // fills issued so far: C buffers, ring slots, per-step objects; items fetched
    int stage, j, t;           // j = step within the item (1..tchunk), t = its T slice
    int cx, y0, z0, pc, zlo, zhi, ylo, yhi, cxlo, cxhi;
    bool done;
    uint64_t pol_n, pol_s, pol_u, pol_p;

    __device__ __forceinline__ void init(const TmaMaps &maps, const TmaParams &prm) {
        tma_prefetch_desc(&maps.psi_c); tma_prefetch_desc(&maps.psi_z); tma_prefetch_desc(&maps.psi_y);
        tma_prefetch_desc(&maps.psi_x); tma_prefetch_desc(&maps.u_c);   tma_prefetch_desc(&maps.u_z);
        tma_prefetch_desc(&maps.u_y);   tma_prefetch_desc(&maps.u_x);   tma_prefetch_desc(&maps.s_c);
        pol_n = l2_policy_evict_normal();
        pol_s = WD_FLAG(prm, 1) ? pol_n : l2_policy_evict_first();  // S is used exactly once
        pol_u = WD_FLAG(prm, 2) ? l2_policy_evict_first() : pol_n;
        pol_p = WD_FLAG(prm, 4) ? l2_policy_evict_last() : pol_n;
        nC = nR = nF = seq = 0;
        stage = ST_FETCH;
        j = t = 0;
        done = false;
    }

    // psi(tt) interior into C buffer nC & 1 (its previous content was fill nC - 2)
    __device__ __forceinline__ bool load_c(const TmaMaps &maps, uint32_t sbase, uint32_t bar_full, uint32_t bar_empty, int tt) {
        const uint32_t b = nC & 1, ob = OB_C + b;
        if (!mbar_try_wait(bar_empty + 8 * ob, ((nC >> 1) & 1) ^ 1)) return false;
        mbar_arrive_expect_tx(bar_full + 8 * ob, P::SZ_C);
        tma_load_5d_hint(sbase + P::OFF_C + b * P::SZ_C, &maps.psi_c, bar_full + 8 * ob, cx, y0, z0, tt, pc, pol_p);
        nC++;
        return true;
    }
    // nine components of U or S into ring slot nR % P::KR (its previous content was fill nR - 4)
    __device__ __forceinline__ bool load_ring(const CUtensorMap *map, uint32_t sbase, uint32_t bar_full, uint32_t bar_empty,
                                              int tt, int comp, uint64_t pol) {
        const uint32_t b = nR % P::KR, ob = OB_R + b;
        if (!mbar_try_wait(bar_empty + 8 * ob, ((nR / P::KR) & 1) ^ 1)) return false;
        mbar_arrive_expect_tx(bar_full + 8 * ob, P::SZ_U);
        tma_load_5d_hint(sbase + P::OFF_R + b * P::SZ_U, map, bar_full + 8 * ob, cx, y0, z0, tt, comp, pol);
        nR++;
        return true;
    }

    __device__ __forceinline__ bool advance(const TmaMaps &maps, const TmaParams &prm, unsigned char *smem, uint32_t sbase,
                                            uint32_t bar_full, uint32_t bar_empty) {
        constexpr int BZ = P::BZ, BY = P::BY, BX = P::BX;
        constexpr bool CLOVER = (P::SELF == SELF_CLOVER);
        if (done) return false;
        const int T = prm.n[0];
        const uint32_t pe = (nF & 1) ^ 1;
        switch (stage) {
        case ST_FETCH: {
            // next work item from the atomic queue, handed to the consumers through a two-slot mailbox
            const uint32_t slot = seq & 1, mpar = (seq >> 1) & 1;
            if (!mbar_try_wait(bar_empty + 8 * (OB_ITEM0 + slot), mpar ^ 1)) return false;
            const int item = fetch_item(prm, seq);
            reinterpret_cast<volatile int *>(smem + P::OFF_MAIL)[slot] = item;
            mbar_arrive(bar_full + 8 * (OB_ITEM0 + slot));
            seq++;
            if (item < 0) {
                done = true;
                return false;
            }
            const Item it = decode_item<P>(prm, item);
            const int Z = prm.n[1], Y = prm.n[2], X = prm.n[3];
            cx = 2 * it.x0, y0 = it.y0, z0 = it.z0;  // dim-0 coordinates count doubles
            pc = 12 * it.rhs0;                       // first component of this right-hand side
            zlo = (z0 == 0) ? Z - 1 : z0 - 1, zhi = (z0 + BZ == Z) ? 0 : z0 + BZ;
            ylo = (y0 == 0) ? Y - 1 : y0 - 1, yhi = (y0 + BY == Y) ? 0 : y0 + BY;
            cxlo = 2 * ((it.x0 == 0) ? X - 1 : it.x0 - 1), cxhi = 2 * ((it.x0 + BX == X) ? 0 : it.x0 + BX);
            t = it.t0;
            j = 1;
            stage = ST_PRO_C;
            return true;
        }
        case ST_PRO_C:  // psi(t0-1) and U_T(t0-1): the backward-T hop of the first slice
            if (!load_c(maps, sbase, bar_full, bar_empty, (t == 0) ? T - 1 : t - 1)) return false;
            stage = ST_PRO_T;
            return true;
        case ST_PRO_T:
            if (!load_ring(&maps.u_c, sbase, bar_full, bar_empty, (t == 0) ? T - 1 : t - 1, 0, pol_u)) return false;
            stage = ST_PRO_C2;
            return true;
        case ST_PRO_C2:  // psi(t0)
            if (!load_c(maps, sbase, bar_full, bar_empty, t)) return false;
            stage = ST_Z;
            return true;
        case ST_Z:
            if (!mbar_try_wait(bar_empty + 8 * OB_Z, pe)) return false;
            mbar_arrive_expect_tx(bar_full + 8 * OB_Z, P::SZ_Z);
            tma_load_5d_hint(sbase + P::OFF_Z, &maps.u_c, bar_full + 8 * OB_Z, cx, y0, z0, t, 9, pol_u);
            tma_load_5d_hint(sbase + P::OFF_ZUF, &maps.u_z, bar_full + 8 * OB_Z, cx, y0, zlo, t, 9, pol_u);
            tma_load_5d_hint(sbase + P::OFF_ZLO, &maps.psi_z, bar_full + 8 * OB_Z, cx, y0, zlo, t, pc, pol_p);
            tma_load_5d_hint(sbase + P::OFF_ZHI, &maps.psi_z, bar_full + 8 * OB_Z, cx, y0, zhi, t, pc, pol_p);
            stage = ST_Y;
            return true;
        case ST_S1:
            if (!load_ring(&maps.s_c, sbase, bar_full, bar_empty, t, 0, pol_s)) return false;
            stage = ST_S2;
            return true;
        case ST_Y:
            if (!mbar_try_wait(bar_empty + 8 * OB_Y, pe)) return false;
            mbar_arrive_expect_tx(bar_full + 8 * OB_Y, P::SZ_Y);
            tma_load_5d_hint(sbase + P::OFF_Y, &maps.u_c, bar_full + 8 * OB_Y, cx, y0, z0, t, 18, pol_u);
            tma_load_5d_hint(sbase + P::OFF_YUF, &maps.u_y, bar_full + 8 * OB_Y, cx, ylo, z0, t, 18, pol_u);
            tma_load_5d_hint(sbase + P::OFF_YLO, &maps.psi_y, bar_full + 8 * OB_Y, cx, ylo, z0, t, pc, pol_p);
            tma_load_5d_hint(sbase + P::OFF_YHI, &maps.psi_y, bar_full + 8 * OB_Y, cx, yhi, z0, t, pc, pol_p);
            stage = CLOVER ? ST_S1 : ST_X;
            return true;
        case ST_S2:
            if (!load_ring(&maps.s_c, sbase, bar_full, bar_empty, t, 9, pol_s)) return false;
            stage = ST_S3;
            return true;
        case ST_X:
            if (!mbar_try_wait(bar_empty + 8 * OB_X, pe)) return false;
            mbar_arrive_expect_tx(bar_full + 8 * OB_X, P::SZ_X);
            tma_load_5d_hint(sbase + P::OFF_X, &maps.u_c, bar_full + 8 * OB_X, cx, y0, z0, t, 27, pol_u);
            tma_load_5d_hint(sbase + P::OFF_XUF, &maps.u_x, bar_full + 8 * OB_X, cxlo, y0, z0, t, 27, pol_u);
            tma_load_5d_hint(sbase + P::OFF_XLO, &maps.psi_x, bar_full + 8 * OB_X, cxlo, y0, z0, t, pc, pol_p);
            tma_load_5d_hint(sbase + P::OFF_XHI, &maps.psi_x, bar_full + 8 * OB_X, cxhi, y0, z0, t, pc, pol_p);
            stage = ST_C;
            return true;
        case ST_S3:
            if (!load_ring(&maps.s_c, sbase, bar_full, bar_empty, t, 18, pol_s)) return false;
            stage = ST_S4;
            return true;
        case ST_S4:
            if (!load_ring(&maps.s_c, sbase, bar_full, bar_empty, t, 27, pol_s)) return false;
            stage = ST_X;
            return true;
        case ST_C:  // psi(t+1): forward-T hop of this slice, then the next step's centre
            if (!load_c(maps, sbase, bar_full, bar_empty, (t + 1 == T) ? 0 : t + 1)) return false;
            stage = ST_T;
            return true;
        default:  // ST_T: U_T(t)
            if (!load_ring(&maps.u_c, sbase, bar_full, bar_empty, t, 0, pol_u)) return false;
            nF++;
            j++;
            t = (t + 1 == T) ? 0 : t + 1;
            stage = (j > prm.tchunk) ? ST_FETCH : ST_Z;
            return true;
        }
    }
};

// ---------------------------------------------------------------- the kernel
// OPEN = false: a periodic lattice — the open-boundary predicates fold away (they cost 9 % more instructions)
template <class P, bool OPEN>
__global__ void __launch_bounds__(P::NTHREADS, 1) k_tma(const __grid_constant__ TmaMaps maps, const TmaParams prm) {
    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t sbase = smem_u32(smem);
    const uint32_t bar_full = sbase + P::OFF_BAR, bar_empty = bar_full + OB_COUNT * 8;
    const int tid = threadIdx.x;
    constexpr int BZ = P::BZ, BY = P::BY, BX = P::BX, N = P::N;
    constexpr bool CLOVER = (P::SELF == SELF_CLOVER);

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
        // ======================= producer: one thread issues every TMA =======================
        if (tid == N) {
            Producer<P> prod;
            prod.init(maps, prm);
            while (!prod.done) prod.advance(maps, prm, smem, sbase, bar_full, bar_empty);
        }
        return;
    }
    // ======================= consumers: one thread per site of the tile =======================
    // The only state a thread carries from phase to phase is acc[12]: the hops of the current slice summed
    // so far, with -2 S psi folded in (out = S psi - 1/2 hops = -1/2 (hops - 2 S psi)).  psi of the own site
    // is re-read from the C buffer where it is needed instead of being kept in registers.
    const int lane = tid & 31;
    const int lx = tid % BX, ly = (tid / BX) % BY, lz = tid / (BX * BY);
    constexpr uint32_t E = P::E, NS = N * E;
    const uint32_t own = tid * E;
    // operand addresses (bytes from the start of shared memory): interior (relative to the C buffer in use)
    // or face storage
    const uint32_t fz = (ly * BX + lx) * E, fy = (lz * BX + lx) * E, fx = (lz * BY + ly) * E;
    const bool zf_in = lz < BZ - 1, zb_in = lz > 0, yf_in = ly < BY - 1, yb_in = ly > 0, xf_in = lx < BX - 1, xb_in = lx > 0;
    const uint32_t z_pf = zf_in ? P::OFF_C + own + P::FZ * E : P::OFF_ZHI + fz, z_pf_s = zf_in ? NS : P::FZ * E;
    const uint32_t z_pb = zb_in ? P::OFF_C + own - P::FZ * E : P::OFF_ZLO + fz, z_b_s = zb_in ? NS : P::FZ * E;
    const uint32_t z_ub = zb_in ? P::OFF_Z + own - P::FZ * E : P::OFF_ZUF + fz;
    const uint32_t y_pf = yf_in ? P::OFF_C + own + BX * E : P::OFF_YHI + fy, y_pf_s = yf_in ? NS : P::FY * E;
    const uint32_t y_pb = yb_in ? P::OFF_C + own - BX * E : P::OFF_YLO + fy, y_b_s = yb_in ? NS : P::FY * E;
    const uint32_t y_ub = yb_in ? P::OFF_Y + own - BX * E : P::OFF_YUF + fy;
    const uint32_t x_pf = xf_in ? P::OFF_C + own + E : P::OFF_XHI + fx, x_pf_s = xf_in ? NS : P::FX * E;
    const uint32_t x_pb = xb_in ? P::OFF_C + own - E : P::OFF_XLO + fx, x_b_s = xb_in ? NS : P::FX * E;
    const uint32_t x_ub = xb_in ? P::OFF_X + own - E : P::OFF_XUF + fx;

    auto release = [&](int ob) {
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8 * ob);
    };
    auto wait_full = [&](int ob, uint32_t parity) { mbar_wait(bar_full + 8 * ob, parity); };

    const long long V = prm.Vs;  // component stride
    const long long strideT = (long long)Z * Y * X;
    uint32_t nC = 0, nR = 0, nF = 0;  // fills consumed so far: C buffers, ring slots, per-step objects
#ifdef WD_EXPERIMENTS
    int ntrace = 0;
#endif
    cd acc[12];

    // own-site psi of C fill n, rows r0..r0+5 scaled by s
    auto load_half = [&](cd q[6], uint32_t cb, int r0, double s) {
#pragma unroll
        for (int c = 0; c < 6; c++) {
            const cd v = lds(smem, P::OFF_C + cb + own + (r0 + c) * NS);
            q[c] = make_double2(s * v.x, s * v.y);
        }
    };
    // one 6x6 block of S (two consecutive ring objects): acc[6b..6b+5] += B_b * (-2 psi)
    auto s_phase = [&](uint32_t cb, int b) {
        const uint32_t s0 = nR % P::KR, s1 = (nR + 1) % P::KR;
        cd q[6];
        load_half(q, cb, 6 * b, -2.0);
        wait_full(OB_R + s0, (nR / P::KR) & 1);
        herm6_half_add<0>(acc + 6 * b, smem, P::OFF_R + s0 * P::SZ_U + own, NS, q);
        wait_full(OB_R + s1, ((nR + 1) / P::KR) & 1);
        herm6_half_add<1>(acc + 6 * b, smem, P::OFF_R + s1 * P::SZ_U + own, NS, q);
        release(OB_R + s0);
        release(OB_R + s1);
        nR += 2;
    };

    const volatile int *mail = reinterpret_cast<const volatile int *>(smem + P::OFF_MAIL);
    for (uint32_t seq = 0;; seq++) {
        const uint32_t mslot = seq & 1, mpar = (seq >> 1) & 1;
        wait_full(OB_ITEM0 + mslot, mpar);
        const int item = mail[mslot];
        release(OB_ITEM0 + mslot);
        if (item < 0) break;
        const Item it = decode_item<P>(prm, item);
        const long long site0 = ((long long)(it.z0 + lz) * Y + (it.y0 + ly)) * X + (it.x0 + lx);
        cd *__restrict__ out = reinterpret_cast<cd *>(prm.out) + (long long)it.rhs0 * 12 * V;
        // open boundaries of a domain-decomposed sub-lattice: hops that would cross them are left out
        const int open = OPEN ? prm.open_mask : 0;
        const bool zf_on = !((open & 2) && it.z0 + lz == Z - 1), zb_on = !((open & 2) && it.z0 + lz == 0);
        const bool yf_on = !((open & 4) && it.y0 + ly == Y - 1), yb_on = !((open & 4) && it.y0 + ly == 0);
        const bool xf_on = !((open & 8) && it.x0 + lx == X - 1), xb_on = !((open & 8) && it.x0 + lx == 0);
        int t = it.t0;
        {   // prologue: acc = backward-T hop of slice t0, (1 + gamma_T) U_T(t0-1)^H psi(t0-1)
            const uint32_t cb = (nC & 1) ? P::SZ_C : 0, slot = nR % P::KR;
            wait_full(OB_C + (nC & 1), (nC >> 1) & 1);
            wait_full(OB_R + slot, (nR / P::KR) & 1);
            cd p[12], u[9], h[6], g[6];
#pragma unroll
            for (int k = 0; k < 9; k++) u[k] = lds(smem, P::OFF_R + slot * P::SZ_U + own + k * NS);
#pragma unroll
            for (int c = 0; c < 12; c++) p[c] = lds(smem, P::OFF_C + cb + own + c * NS);
            release(OB_C + (nC & 1));
            release(OB_R + slot);
            nC++;
            nR++;
            project<0, +1>(h, p);
            su3_mul<true>(g, u, h);
#pragma unroll
            for (int c = 0; c < 12; c++) acc[c] = make_double2(0.0, 0.0);
            if (!((open & 1) && it.t0 == 0)) reconstruct_add<0, +1>(acc, g);
        }
        for (int j = 1; j <= prm.tchunk; j++) {
            const bool last = (j == prm.tchunk);
            const uint32_t cb = (nC & 1) ? P::SZ_C : 0;  // C buffer holding psi(t) (waited for at the end of the
            if (j == 1) wait_full(OB_C + (nC & 1), (nC >> 1) & 1);  // previous step, except for the first slice)
            const uint32_t pf = nF & 1;
            wait_full(OB_Z, pf);
            hop_pair_smem<1>(acc, smem, P::OFF_Z + own, NS, z_pf + (zf_in ? cb : 0), z_pf_s, z_ub, z_b_s,
                             z_pb + (zb_in ? cb : 0), z_b_s, zf_on, zb_on);
            release(OB_Z);
            wait_full(OB_Y, pf);
            hop_pair_smem<2>(acc, smem, P::OFF_Y + own, NS, y_pf + (yf_in ? cb : 0), y_pf_s, y_ub, y_b_s,
                             y_pb + (yb_in ? cb : 0), y_b_s, yf_on, yb_on);
            release(OB_Y);
            if (CLOVER) {  // between the Y and X hops, so that neither S4 nor the next U_T waits on a just-freed slot
                s_phase(cb, 0);
                s_phase(cb, 1);
            }
            wait_full(OB_X, pf);
            hop_pair_smem<3>(acc, smem, P::OFF_X + own, NS, x_pf + (xf_in ? cb : 0), x_pf_s, x_ub, x_b_s,
                             x_pb + (xb_in ? cb : 0), x_b_s, xf_on, xb_on);
            release(OB_X);
            nF++;
            {   // T phase: forward hop (1 - gamma_T) U_T(t) psi(t+1) completes out(t); the backward hop of slice
                // t+1, (1 + gamma_T) U_T(t)^H psi(t), starts the next accumulator
                const uint32_t cn = cb ^ P::SZ_C, slot = nR % P::KR;  // psi(t+1) is in the other C buffer
                wait_full(OB_C + ((nC + 1) & 1), ((nC + 1) >> 1) & 1);
                wait_full(OB_R + slot, (nR / P::KR) & 1);
#ifdef WD_EXPERIMENTS
                if (prm.trace && tid == 0 && ntrace < kTraceLen) {
                    unsigned long long now;
                    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(now));
                    prm.trace[(size_t)blockIdx.x * kTraceLen + ntrace++] = now;
                }
#endif
                cd u[9], p[12];
#pragma unroll
                for (int k = 0; k < 9; k++) u[k] = lds(smem, P::OFF_R + slot * P::SZ_U + own + k * NS);
#pragma unroll
                for (int c = 0; c < 12; c++) p[c] = lds(smem, P::OFF_C + cn + own + c * NS);
                if (!((open & 1) && t == T - 1)) hop_term<0, -1>(acc, p, u);
                if (P::SELF == SELF_MASS || !last) {
#pragma unroll
                    for (int c = 0; c < 12; c++) p[c] = lds(smem, P::OFF_C + cb + own + c * NS);  // psi(t)
                }
                const long long ip = (long long)t * strideT + site0;
#pragma unroll
                for (int c = 0; c < 12; c++) {
                    cd o = make_double2(-0.5 * acc[c].x, -0.5 * acc[c].y);
                    if (P::SELF == SELF_MASS) o = make_double2(fma(prm.mass, p[c].x, o.x), fma(prm.mass, p[c].y, o.y));
                    __stcs(out + (long long)c * V + ip, o);
                }
                if (!last) {
                    cd h[6], g[6];
                    project<0, +1>(h, p);
                    su3_mul<true>(g, u, h);
                    reconstruct_set<0, +1>(acc, g);
                }
                release(OB_R + slot);
                nR++;
                release(OB_C + (nC & 1));  // psi(t) is done; psi(t+1) stays for the next step
                nC++;
                if (last) {                // ... unless this was the item's last slice
                    release(OB_C + (nC & 1));
                    nC++;
                }
            }
            t = (t + 1 == T) ? 0 : t + 1;
        }
    }
}

// ---------------------------------------------------------------- host side
// Short chunks keep the CTAs of a panel within a few steps of each other (each item starts at a chunk boundary),
// which is what makes the face re-reads L2 hits; the price is one extra psi and U_T slice per item.  Measured at
// 64^4: tchunk 8 and 16 beat 32 and 64 by 3-7 % (CHUNK_SHORT).
template <int BZ, int BY, int BX, int SELF, int KR> static cudaError_t launch_tma_self(const KParams &p, cudaStream_t st) {
    using P = Plan<BZ, BY, BX, SELF, KR>;
    // 8-site rows (4x4x8, 2x8x8): short chunks; the 2x4x16 tile does better with the cost model (64^4 Wilson: 2.83 vs 2.87 ms)
    const ChunkPolicy pol = (BX >= 16) ? CHUNK_COST_MODEL : CHUNK_SHORT;
    return p.open_mask ? launch_tma_kernel<P>(k_tma<P, true>, p, st, /*ucomp*/ 9, /*scomp*/ 9, pol, /*rb*/ 4) : launch_tma_kernel<P>(k_tma<P, false>, p, st, /*ucomp*/ 9, /*scomp*/ 9, pol, /*rb*/ 4);
}

template <int BZ, int BY, int BX, int KR = 4> static cudaError_t launch_tma(const KParams &p, int self, cudaStream_t st) {
    if (self == SELF_CLOVER) return launch_tma_self<BZ, BY, BX, SELF_CLOVER, KR>(p, st);
    if (self == SELF_MASS) return launch_tma_self<BZ, BY, BX, SELF_MASS, KR>(p, st);
    return launch_tma_self<BZ, BY, BX, SELF_NONE, KR>(p, st);
}
}  // namespace tmb

// Tiles of 128 sites whose shared-memory plan fits 227 KB (2x4x16 is 816 B too large)
cudaError_t launch_tmb_4x4x8(const KParams &p, int self, cudaStream_t st) { return tmb::launch_tma<4, 4, 8>(p, self, st); }
cudaError_t launch_tmb_2x4x16(const KParams &p, int self, cudaStream_t st) { return tmb::launch_tma<2, 4, 16, 3>(p, self, st); }
}  // namespace wd
