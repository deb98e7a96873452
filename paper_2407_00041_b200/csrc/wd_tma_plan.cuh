// wd_tma_plan.cuh — the shared-memory plan and the producer of the first-generation TMA kernel, shared by wd_tma.cu
// (one compute warpgroup per tile; FP64, two-row links, FP32) and wd_tmw.cu (two compute warpgroups per tile).
#pragma once
#include "wd_tma_common.cuh"
#include "wd_smem_ops.cuh"

namespace wd {
namespace gen1 {

// ---------------------------------------------------------------- shared-memory plan
// Objects (each with a full/empty mbarrier pair), refilled once per T step:
//   C  psi(t) interior                                    [12][N]
//   T  U_T(t-1) interior                                  [9][N]
//   Z  U_Z(t) interior | U_Z face z0-1 | psi faces z0-1, z0+BZ      [9][N] [9][FZ] [12][FZ] [12][FZ]
//   Y  same for Y;  X  same for X
//   SA, SB  the two 6x6 blocks of S(t)                    [18][N] each
enum { OB_C = 0, OB_T, OB_Z, OB_Y, OB_X, OB_SA };  // then OB_SB, OB_ITEM0, OB_ITEM1 (work-item mailbox): see Plan

// UC = complex numbers stored per link: 9, or 6 with two-row storage (WD_OPT_GAUGE_ROWS = 2: the third row of an SU(3)
// link is the conjugate cross product of the first two and is rebuilt in registers, wd_smem_ops.cuh)
// C = complex element type: double2 (FP64) or float2 (the FP32 variant, wd_f32.cu).  Sub-objects are padded to 128
// bytes, the alignment TMA needs for a shared-memory destination (only the 8-byte X link face is not a multiple already).
constexpr uint32_t al128(uint32_t x) { return (x + 127u) & ~127u; }
template <int BZ_, int BY_, int BX_, int SELF_, int UC_ = 9, class C_ = cd> struct Plan {
    typedef C_ C;
    static constexpr int BZ = BZ_, BY = BY_, BX = BX_, SELF = SELF_, UC = UC_;
    static constexpr int G = 1;             // right-hand sides per work item
    static constexpr bool BLK = false;      // plain multi-RHS layout only (the quad kernels of wd_tmq.cu read the blocked one)
    static constexpr int RBK = 1;
    static constexpr int N = BZ * BY * BX;  // sites per tile = compute threads
    static constexpr int NW = N / 32;       // compute warps
    static constexpr int NTHREADS = N + 32; // + the producer warp
    static constexpr uint32_t E = sizeof(C);                        // bytes per element
    // A TMA box must be a multiple of 16 bytes wide: the X faces of 8-byte elements are fetched two sites wide (the
    // neighbour column and the one beyond it), of which the consumers read one.
    static constexpr int XW = (E == 8) ? 2 : 1;

    static constexpr int FZ = BY * BX, FY = BZ * BX, FX = BZ * BY * XW;  // sites stored per face
    static constexpr uint32_t SZ_C = 12 * N * E, SZ_U = UC * N * E, SZ_S = 18 * N * E;
    static constexpr uint32_t OFF_C = 0;
    static constexpr uint32_t OFF_T = OFF_C + SZ_C;
    static constexpr uint32_t OFF_Z = OFF_T + SZ_U;
    static constexpr uint32_t OFF_ZUF = OFF_Z + SZ_U, OFF_ZLO = OFF_ZUF + al128(UC * FZ * E), OFF_ZHI = OFF_ZLO + 12 * FZ * E;
    static constexpr uint32_t SZ_Z = SZ_U + (UC + 24) * FZ * E;  // bytes the TMA delivers
    static constexpr uint32_t SP_Z = SZ_U + al128(UC * FZ * E) + 24 * FZ * E;  // bytes it occupies
    static constexpr uint32_t OFF_Y = OFF_Z + SP_Z;
    static constexpr uint32_t OFF_YUF = OFF_Y + SZ_U, OFF_YLO = OFF_YUF + al128(UC * FY * E), OFF_YHI = OFF_YLO + 12 * FY * E;
    static constexpr uint32_t SZ_Y = SZ_U + (UC + 24) * FY * E;  // bytes the TMA delivers
    static constexpr uint32_t SP_Y = SZ_U + al128(UC * FY * E) + 24 * FY * E;  // bytes it occupies
    static constexpr uint32_t OFF_X = OFF_Y + SP_Y;
    static constexpr uint32_t OFF_XUF = OFF_X + SZ_U, OFF_XLO = OFF_XUF + al128(UC * FX * E), OFF_XHI = OFF_XLO + 12 * FX * E;
    static constexpr uint32_t SZ_X = SZ_U + (UC + 24) * FX * E;  // bytes the TMA delivers
    static constexpr uint32_t SP_X = SZ_U + al128(UC * FX * E) + 24 * FX * E;  // bytes it occupies
    static constexpr uint32_t OFF_SA = OFF_X + SP_X;
    static constexpr uint32_t OFF_SB = OFF_SA + SZ_S;
    static constexpr uint32_t OFF_BAR = (SELF == SELF_CLOVER) ? OFF_SB + SZ_S : OFF_SA;
    // COMPACT (8-byte elements with S): the two blocks of S share one barrier pair and the mailbox has one slot, which
    // brings the plan to 115 704 B — two CTAs (8 compute warps) per SM; measured on the FP32 Wilson kernel: 2.45 -> 1.93 ms
    static constexpr bool COMPACT = (E == 8) && (SELF == SELF_CLOVER);
    static constexpr int OB_SB = COMPACT ? OB_SA : OB_SA + 1;
    static constexpr int OB_ITEM0 = OB_SB + 1, OB_ITEM1 = COMPACT ? OB_ITEM0 : OB_ITEM0 + 1;
    static constexpr int OB_COUNT = OB_ITEM1 + 1;
    static constexpr uint32_t OFF_MAIL = OFF_BAR + 2 * OB_COUNT * 8;  // int per mailbox slot: item index
    static constexpr uint32_t SMEM = OFF_MAIL + (COMPACT ? 8 : 16);
    // persistent CTAs per SM: two (8 compute warps) where two plans plus the 1 KB the system reserves per CTA fit the
    // 228 KB of an SM — the plans of 8-byte elements without S buffers
    static constexpr int CTAS_PER_SM = (2 * (SMEM + 1024) <= 233472) ? 2 : 1;
    static_assert(N % 32 == 0 && (12 * FZ * E) % 128 == 0 && (12 * FY * E) % 128 == 0 && (12 * FX * E) % 128 == 0 && SZ_U % 128 == 0,
                  "tile faces must keep 128-byte alignment");
    static_assert(SMEM <= 232448, "shared-memory plan exceeds 227 KB");
};

// ---------------------------------------------------------------- the producer (one thread)
// Streams everything a tile needs, object by object, each guarded by a full/empty mbarrier pair.  Per step the order
// is the order in which the consumers release the buffers of the previous step: T, Z, Y, X, psi, S_A, S_B — with
// Y_LAST (wd_tmw.cu, whose Y buffer doubles as the hand-over buffer of the two warpgroups): T, Z, X, psi, S_A, S_B, Y.
template <class P, bool Y_LAST>
__device__ __forceinline__ void producer(const TmaMaps &maps, const TmaParams &prm, unsigned char *smem, uint32_t sbase,
                                         uint32_t bar_full, uint32_t bar_empty) {
    constexpr int BZ = P::BZ, BY = P::BY, BX = P::BX;
    constexpr bool CLOVER = (P::SELF == SELF_CLOVER);
    constexpr int OB_SB = P::OB_SB, OB_ITEM0 = P::OB_ITEM0;
    const int T = prm.n[0], Z = prm.n[1], Y = prm.n[2], X = prm.n[3];
    tma_prefetch_desc(&maps.psi_c); tma_prefetch_desc(&maps.psi_z); tma_prefetch_desc(&maps.psi_y);
    tma_prefetch_desc(&maps.psi_x); tma_prefetch_desc(&maps.u_c);   tma_prefetch_desc(&maps.u_z);
    tma_prefetch_desc(&maps.u_y);   tma_prefetch_desc(&maps.u_x);   tma_prefetch_desc(&maps.s_c);
    const uint64_t pol_n = l2_policy_evict_normal();
    const uint64_t pol_s = WD_FLAG(prm, 1) ? pol_n : l2_policy_evict_first();  // S is used exactly once
    const uint64_t pol_u = WD_FLAG(prm, 2) ? l2_policy_evict_first() : pol_n;
    const uint64_t pol_p = WD_FLAG(prm, 4) ? l2_policy_evict_last() : pol_n;
    uint32_t nC = 0, nT = 0, nF = 0;  // fills issued so far of C, T, and of the per-step objects
    volatile int *mail = reinterpret_cast<volatile int *>(smem + P::OFF_MAIL);
    for (uint32_t seq = 0;; seq++) {
        // next work item from the atomic queue, handed to the consumers through a two-slot mailbox
        const int item = fetch_item(prm, seq);
        const uint32_t slot = P::COMPACT ? 0 : (seq & 1), mpar = P::COMPACT ? (seq & 1) : ((seq >> 1) & 1);
        mbar_wait(bar_empty + 8 * (OB_ITEM0 + slot), mpar ^ 1);
        mail[slot] = item;
        mbar_arrive(bar_full + 8 * (OB_ITEM0 + slot));
        if (item < 0) break;
        const Item it = decode_item<P>(prm, item);
        const int cx = 2 * it.x0, y0 = it.y0, z0 = it.z0;  // dim-0 coordinates count real numbers
        const int pc = 12 * it.rhs0;                       // first component of this right-hand side
        const int zlo = (z0 == 0) ? Z - 1 : z0 - 1, zhi = (z0 + BZ == Z) ? 0 : z0 + BZ;
        const int ylo = (y0 == 0) ? Y - 1 : y0 - 1, yhi = (y0 + BY == Y) ? 0 : y0 + BY;
        const int cxlo = 2 * ((it.x0 == 0) ? X - P::XW : it.x0 - P::XW), cxhi = 2 * ((it.x0 + BX == X) ? 0 : it.x0 + BX);
        int t = (it.t0 == 0) ? T - 1 : it.t0 - 1;
        // prologue: psi(t0-1), only to seed the carried half-spinor
        mbar_wait(bar_empty + 8 * OB_C, (nC & 1) ^ 1);
        mbar_arrive_expect_tx(bar_full + 8 * OB_C, P::SZ_C);
        tma_load_5d_hint(sbase + P::OFF_C, &maps.psi_c, bar_full + 8 * OB_C, cx, y0, z0, t, pc, pol_p);
        nC++;
        for (int j = 1; j <= prm.tchunk + 1; j++) {
            const int tprev = t;
            t = (t + 1 == T) ? 0 : t + 1;
            const bool full = (j <= prm.tchunk);
            // T object: U_T(t-1)
            mbar_wait(bar_empty + 8 * OB_T, (nT & 1) ^ 1);
            mbar_arrive_expect_tx(bar_full + 8 * OB_T, P::SZ_U);
            tma_load_5d_hint(sbase + P::OFF_T, &maps.u_c, bar_full + 8 * OB_T, cx, y0, z0, tprev, 0, pol_u);
            nT++;
            if (full) {
                const uint32_t pe = (nF & 1) ^ 1;
                mbar_wait(bar_empty + 8 * OB_Z, pe);
                mbar_arrive_expect_tx(bar_full + 8 * OB_Z, P::SZ_Z);
                tma_load_5d_hint(sbase + P::OFF_Z, &maps.u_c, bar_full + 8 * OB_Z, cx, y0, z0, t, P::UC, pol_u);
                tma_load_5d_hint(sbase + P::OFF_ZUF, &maps.u_z, bar_full + 8 * OB_Z, cx, y0, zlo, t, P::UC, pol_u);
                tma_load_5d_hint(sbase + P::OFF_ZLO, &maps.psi_z, bar_full + 8 * OB_Z, cx, y0, zlo, t, pc, pol_p);
                tma_load_5d_hint(sbase + P::OFF_ZHI, &maps.psi_z, bar_full + 8 * OB_Z, cx, y0, zhi, t, pc, pol_p);
                if (!Y_LAST) {
                    mbar_wait(bar_empty + 8 * OB_Y, pe);
                    mbar_arrive_expect_tx(bar_full + 8 * OB_Y, P::SZ_Y);
                    tma_load_5d_hint(sbase + P::OFF_Y, &maps.u_c, bar_full + 8 * OB_Y, cx, y0, z0, t, 2 * P::UC, pol_u);
                    tma_load_5d_hint(sbase + P::OFF_YUF, &maps.u_y, bar_full + 8 * OB_Y, cx, ylo, z0, t, 2 * P::UC, pol_u);
                    tma_load_5d_hint(sbase + P::OFF_YLO, &maps.psi_y, bar_full + 8 * OB_Y, cx, ylo, z0, t, pc, pol_p);
                    tma_load_5d_hint(sbase + P::OFF_YHI, &maps.psi_y, bar_full + 8 * OB_Y, cx, yhi, z0, t, pc, pol_p);
                }
                mbar_wait(bar_empty + 8 * OB_X, pe);
                mbar_arrive_expect_tx(bar_full + 8 * OB_X, P::SZ_X);
                tma_load_5d_hint(sbase + P::OFF_X, &maps.u_c, bar_full + 8 * OB_X, cx, y0, z0, t, 3 * P::UC, pol_u);
                tma_load_5d_hint(sbase + P::OFF_XUF, &maps.u_x, bar_full + 8 * OB_X, cxlo, y0, z0, t, 3 * P::UC, pol_u);
                tma_load_5d_hint(sbase + P::OFF_XLO, &maps.psi_x, bar_full + 8 * OB_X, cxlo, y0, z0, t, pc, pol_p);
                tma_load_5d_hint(sbase + P::OFF_XHI, &maps.psi_x, bar_full + 8 * OB_X, cxhi, y0, z0, t, pc, pol_p);
            }
            // C object: psi(t).  Its buffer is released after the X phase of the previous step, so it
            // has only the S phases to land.  (Warming L2 one step ahead with a TMA prefetch was
            // measured to cost 20 % at 64^4 — flag 8, profiles/r1b — so it is off.)
            mbar_wait(bar_empty + 8 * OB_C, (nC & 1) ^ 1);
            mbar_arrive_expect_tx(bar_full + 8 * OB_C, P::SZ_C);
            tma_load_5d_hint(sbase + P::OFF_C, &maps.psi_c, bar_full + 8 * OB_C, cx, y0, z0, t, pc, pol_p);
            nC++;
            if (full && WD_FLAG(prm, 8)) tma_prefetch_5d(&maps.psi_c, cx, y0, z0, (t + 1 == T) ? 0 : t + 1, pc);
            if (full && CLOVER) {
                const uint32_t pe = (nF & 1) ^ 1;
                mbar_wait(bar_empty + 8 * OB_SA, pe);
                mbar_arrive_expect_tx(bar_full + 8 * OB_SA, P::COMPACT ? 2 * P::SZ_S : P::SZ_S);
                tma_load_5d_hint(sbase + P::OFF_SA, &maps.s_c, bar_full + 8 * OB_SA, cx, y0, z0, t, 0, pol_s);
                if (!P::COMPACT) {
                    mbar_wait(bar_empty + 8 * OB_SB, pe);
                    mbar_arrive_expect_tx(bar_full + 8 * OB_SB, P::SZ_S);
                }
                tma_load_5d_hint(sbase + P::OFF_SB, &maps.s_c, bar_full + 8 * OB_SB, cx, y0, z0, t, 18, pol_s);
            }
            if (full && Y_LAST) {  // its buffer comes back last (wd_tmw.cu: after the hand-over of the previous step)
                const uint32_t pe = (nF & 1) ^ 1;
                mbar_wait(bar_empty + 8 * OB_Y, pe);
                mbar_arrive_expect_tx(bar_full + 8 * OB_Y, P::SZ_Y);
                tma_load_5d_hint(sbase + P::OFF_Y, &maps.u_c, bar_full + 8 * OB_Y, cx, y0, z0, t, 2 * P::UC, pol_u);
                tma_load_5d_hint(sbase + P::OFF_YUF, &maps.u_y, bar_full + 8 * OB_Y, cx, ylo, z0, t, 2 * P::UC, pol_u);
                tma_load_5d_hint(sbase + P::OFF_YLO, &maps.psi_y, bar_full + 8 * OB_Y, cx, ylo, z0, t, pc, pol_p);
                tma_load_5d_hint(sbase + P::OFF_YHI, &maps.psi_y, bar_full + 8 * OB_Y, cx, yhi, z0, t, pc, pol_p);
            }
            if (full) nF++;
        }
    }
}

}  // namespace gen1
}  // namespace wd
