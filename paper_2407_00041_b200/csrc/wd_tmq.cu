// wd_tmq.cu — the "quad" kernels for several right-hand sides in one call (a8; multi-tuple
// reads): one compute thread per (site, right-hand side), G = 4 right-hand sides per work item.
//
// The multi-RHS runs of the one-thread-per-site TMA kernels are bound by the shared-memory pipe, not by HBM: every
// right-hand side stages and reads its own copy of the links and of S (profiles/r1c, r2).  Here a work item is a 64-site
// tile x 4 right-hand sides: 256 compute threads (two warpgroups at 232 registers, the producer warpgroup gives its share
// away with setmaxnreg), the links and S of the tile come through L2 and shared memory ONCE for the four, and the four
// threads of a site read them with one address.
//   tmq_*   plain multi-RHS layout  double2 [nrhs][12][Vs]:       lane = r * 8 + site; psi boxes [r][component][site]
//   tmqb_*  blocked layout (WD_OPT_RHS_BLOCK = 4)  [unit][12][Vs][4]: lane = site * 4 + r; psi boxes [component][site][r];
//           a warp reads 512 consecutive bytes per psi component (four conflict-free wavefronts), and an LDS.128 of a
//           link or S entry — one address per four adjacent lanes — costs two wavefronts instead of four.  (Measured on
//           B200: the pipe merges quarter-warps only when their banks are disjoint, so the lane = r * 8 + site pattern of
//           the plain layout, whose quarter-warps read the same 128 bytes, still pays four.)
// Skeleton = first generation (wd_tma.cu): persistent CTA, one producer thread, objects with full/empty mbarrier pairs,
// T-marching with the T hops carried in registers.  What differs, because psi is now four times as large as the links:
//   * psi(t) interior is DOUBLE-buffered: psi(t+2) is requested as soon as the Z phase of step t has released psi(t), a
//     full step before its first use.  (Single-buffered, the 49 KB box had only the S phases to arrive from HBM and the
//     consumers spent 18 % of all issue slots waiting for it, profiles/r2_prof_tmqb_*.)
//   * the two 6x6 blocks of S have no buffers of their own: S_A lands in the X object's buffer once the X hops are done,
//     S_B in the Y object's, and the phase order is T, X, Y, Z, S_A, S_B — that is what makes room for the second psi
//     buffer (229 KB in all).
#include <cstdio>
#include <cstdlib>

#include "wd_smem_ops.cuh"
#include "wd_tma_common.cuh"

namespace wd {
namespace tmq {

// ---------------------------------------------------------------- shared-memory plan
// Objects (each with a full/empty mbarrier pair):
//   C0, C1  psi interior of two consecutive slices (fill n in buffer n & 1)      [12 G][N] elements
//   T       U_T(t-1) interior                                                     [9][N]
//   RX      alternately  X(t): U_X(t) interior | U_X face x0-1 | psi faces x0-1, x0+BX    and  S_A(t): [18][N]
//   RY      alternately  Y(t) (same for Y)  and  S_B(t)
//   RZ      Z(t)
enum { OB_C0 = 0, OB_C1, OB_T, OB_RX, OB_RY, OB_RZ, OB_ITEM0, OB_ITEM1, OB_COUNT };

constexpr uint32_t al128(uint32_t x) { return (x + 127u) & ~127u; }

template <int BZ_, int BY_, int BX_, int SELF_, bool BLK_> struct Plan {
    typedef cd C;
    static constexpr int BZ = BZ_, BY = BY_, BX = BX_, SELF = SELF_;
    static constexpr int G = 4;                  // right-hand sides per work item
    static constexpr bool BLK = BLK_;            // blocked multi-RHS layout
    static constexpr int RBK = BLK ? G : 1;      // right-hand sides interleaved per site in the spinor fields
    static constexpr int N = BZ * BY * BX;       // sites per tile
    static constexpr int NC = N * G;             // compute threads
    static constexpr int NW = NC / 32;           // compute warps
    static constexpr int NTHREADS = NC + 128;    // + the producer's warpgroup (setmaxnreg works on whole warpgroups)
    static constexpr int CTAS_PER_SM = 1;
    static constexpr int XW = 1;
    static constexpr int PC = 12 * G;            // spinor components per box
    static constexpr int FZ = BY * BX, FY = BZ * BX, FX = BZ * BY;  // sites per face
    static constexpr uint32_t E = 16;
    static constexpr uint32_t SZ_C = PC * N * E, SZ_U = 9 * N * E, SZ_S = 18 * N * E;
    static constexpr uint32_t OFF_C = 0;
    static constexpr uint32_t OFF_T = OFF_C + 2 * SZ_C;
    static constexpr uint32_t OFF_X = OFF_T + SZ_U;
    static constexpr uint32_t OFF_XUF = OFF_X + SZ_U, OFF_XLO = OFF_XUF + al128(9 * FX * E), OFF_XHI = OFF_XLO + PC * FX * E;
    static constexpr uint32_t SZ_X = SZ_U + (9 + 2 * PC) * FX * E;            // bytes the TMA delivers
    static constexpr uint32_t SP_X = SZ_U + al128(9 * FX * E) + 2 * PC * FX * E;  // bytes the object occupies
    static constexpr uint32_t OFF_Y = OFF_X + SP_X;
    static constexpr uint32_t OFF_YUF = OFF_Y + SZ_U, OFF_YLO = OFF_YUF + al128(9 * FY * E), OFF_YHI = OFF_YLO + PC * FY * E;
    static constexpr uint32_t SZ_Y = SZ_U + (9 + 2 * PC) * FY * E;
    static constexpr uint32_t SP_Y = SZ_U + al128(9 * FY * E) + 2 * PC * FY * E;
    static constexpr uint32_t OFF_Z = OFF_Y + SP_Y;
    static constexpr uint32_t OFF_ZUF = OFF_Z + SZ_U, OFF_ZLO = OFF_ZUF + al128(9 * FZ * E), OFF_ZHI = OFF_ZLO + PC * FZ * E;
    static constexpr uint32_t SZ_Z = SZ_U + (9 + 2 * PC) * FZ * E;
    static constexpr uint32_t SP_Z = SZ_U + al128(9 * FZ * E) + 2 * PC * FZ * E;
    static constexpr uint32_t OFF_BAR = OFF_Z + SP_Z;
    static constexpr uint32_t OFF_MAIL = OFF_BAR + 2 * OB_COUNT * 8;
    static constexpr uint32_t SMEM = OFF_MAIL + 16;
    static_assert(NC == 256, "two compute warpgroups");
    static_assert(SZ_S <= SP_X && SZ_S <= SP_Y, "a block of S must fit the X and Y objects' buffers");
    static_assert((PC * FZ * E) % 128 == 0 && (PC * FY * E) % 128 == 0 && (PC * FX * E) % 128 == 0 && SZ_U % 128 == 0, "TMA destinations need 128-byte alignment");
    static_assert(SMEM <= 232448, "shared-memory plan exceeds 227 KB");
};

// ---------------------------------------------------------------- the producer (one thread)
// Issues every load in the order in which the consumers free its destination.  Steady state, while the consumers are in
// step j (slice t) of an item:  U_T(t) -> T (after their T phase) | S_A(t) -> RX (after the X hops) | S_B(t) -> RY (after
// the Y hops) | Z(t+1) -> RZ and psi(t+2) -> the buffer of psi(t) (after the Z hops) | X(t+1) -> RX (after S_A) | Y(t+1) ->
// RY (after S_B).
template <class P>
__device__ __forceinline__ void producer(const TmaMaps &maps, const TmaParams &prm, unsigned char *smem, uint32_t sbase,
                                         uint32_t bar_full, uint32_t bar_empty) {
    constexpr int BZ = P::BZ, BY = P::BY, BX = P::BX, RBK = P::RBK;
    constexpr bool CLOVER = (P::SELF == SELF_CLOVER);
    const int T = prm.n[0], Z = prm.n[1], Y = prm.n[2], X = prm.n[3];
    tma_prefetch_desc(&maps.psi_c); tma_prefetch_desc(&maps.psi_z); tma_prefetch_desc(&maps.psi_y);
    tma_prefetch_desc(&maps.psi_x); tma_prefetch_desc(&maps.u_c);   tma_prefetch_desc(&maps.u_z);
    tma_prefetch_desc(&maps.u_y);   tma_prefetch_desc(&maps.u_x);   tma_prefetch_desc(&maps.s_c);
    const uint64_t pol_n = l2_policy_evict_normal();
    // S and the links serve the other units of the tile from L2 (item order: wd_tma_common.cuh): default policy
    uint32_t nC = 0, nT = 0, nX = 0, nY = 0, nZ = 0;  // fills issued so far
    volatile int *mail = reinterpret_cast<volatile int *>(smem + P::OFF_MAIL);
    for (uint32_t seq = 0;; seq++) {
        const int item = fetch_item(prm, seq);
        const uint32_t slot = seq & 1, mpar = (seq >> 1) & 1;
        mbar_wait(bar_empty + 8 * (OB_ITEM0 + slot), mpar ^ 1);
        mail[slot] = item;
        mbar_arrive(bar_full + 8 * (OB_ITEM0 + slot));
        if (item < 0) break;
        const Item it = decode_item<P>(prm, item);
        const int cx = 2 * it.x0, y0 = it.y0, z0 = it.z0;  // dim-0 coordinates count real numbers
        const int pc = P::BLK ? 12 * (it.rhs0 / P::G) : 12 * it.rhs0;  // first spinor component of the unit
        const int zlo = (z0 == 0) ? Z - 1 : z0 - 1, zhi = (z0 + BZ == Z) ? 0 : z0 + BZ;
        const int ylo = (y0 == 0) ? Y - 1 : y0 - 1, yhi = (y0 + BY == Y) ? 0 : y0 + BY;
        const int cxlo = 2 * ((it.x0 == 0) ? X - 1 : it.x0 - 1), cxhi = 2 * ((it.x0 + BX == X) ? 0 : it.x0 + BX);
        const int cxp = RBK * cx, cxplo = RBK * cxlo, cxphi = RBK * cxhi;  // spinor boxes: 2 RBK reals per site

        auto load_c = [&](int tt) {  // psi(tt) interior into buffer nC & 1
            const uint32_t b = nC & 1;
            mbar_wait(bar_empty + 8 * (OB_C0 + b), ((nC >> 1) & 1) ^ 1);
            mbar_arrive_expect_tx(bar_full + 8 * (OB_C0 + b), P::SZ_C);
            tma_load_5d_hint(sbase + P::OFF_C + b * P::SZ_C, &maps.psi_c, bar_full + 8 * (OB_C0 + b), cxp, y0, z0, tt, pc, pol_n);
            nC++;
        };
        auto load_t = [&](int tt) {  // U_T(tt)
            mbar_wait(bar_empty + 8 * OB_T, (nT & 1) ^ 1);
            mbar_arrive_expect_tx(bar_full + 8 * OB_T, P::SZ_U);
            tma_load_5d_hint(sbase + P::OFF_T, &maps.u_c, bar_full + 8 * OB_T, cx, y0, z0, tt, 0, pol_n);
            nT++;
        };
        auto load_x = [&](int tt) {
            mbar_wait(bar_empty + 8 * OB_RX, (nX & 1) ^ 1);
            mbar_arrive_expect_tx(bar_full + 8 * OB_RX, P::SZ_X);
            tma_load_5d_hint(sbase + P::OFF_X, &maps.u_c, bar_full + 8 * OB_RX, cx, y0, z0, tt, 27, pol_n);
            tma_load_5d_hint(sbase + P::OFF_XUF, &maps.u_x, bar_full + 8 * OB_RX, cxlo, y0, z0, tt, 27, pol_n);
            tma_load_5d_hint(sbase + P::OFF_XLO, &maps.psi_x, bar_full + 8 * OB_RX, cxplo, y0, z0, tt, pc, pol_n);
            tma_load_5d_hint(sbase + P::OFF_XHI, &maps.psi_x, bar_full + 8 * OB_RX, cxphi, y0, z0, tt, pc, pol_n);
            nX++;
        };
        auto load_y = [&](int tt) {
            mbar_wait(bar_empty + 8 * OB_RY, (nY & 1) ^ 1);
            mbar_arrive_expect_tx(bar_full + 8 * OB_RY, P::SZ_Y);
            tma_load_5d_hint(sbase + P::OFF_Y, &maps.u_c, bar_full + 8 * OB_RY, cx, y0, z0, tt, 18, pol_n);
            tma_load_5d_hint(sbase + P::OFF_YUF, &maps.u_y, bar_full + 8 * OB_RY, cx, ylo, z0, tt, 18, pol_n);
            tma_load_5d_hint(sbase + P::OFF_YLO, &maps.psi_y, bar_full + 8 * OB_RY, cxp, ylo, z0, tt, pc, pol_n);
            tma_load_5d_hint(sbase + P::OFF_YHI, &maps.psi_y, bar_full + 8 * OB_RY, cxp, yhi, z0, tt, pc, pol_n);
            nY++;
        };
        auto load_z = [&](int tt) {
            mbar_wait(bar_empty + 8 * OB_RZ, (nZ & 1) ^ 1);
            mbar_arrive_expect_tx(bar_full + 8 * OB_RZ, P::SZ_Z);
            tma_load_5d_hint(sbase + P::OFF_Z, &maps.u_c, bar_full + 8 * OB_RZ, cx, y0, z0, tt, 9, pol_n);
            tma_load_5d_hint(sbase + P::OFF_ZUF, &maps.u_z, bar_full + 8 * OB_RZ, cx, y0, zlo, tt, 9, pol_n);
            tma_load_5d_hint(sbase + P::OFF_ZLO, &maps.psi_z, bar_full + 8 * OB_RZ, cxp, y0, zlo, tt, pc, pol_n);
            tma_load_5d_hint(sbase + P::OFF_ZHI, &maps.psi_z, bar_full + 8 * OB_RZ, cxp, y0, zhi, tt, pc, pol_n);
            nZ++;
        };
        auto load_sa = [&](int tt) {  // block A of S(tt) into the X object's buffer
            mbar_wait(bar_empty + 8 * OB_RX, (nX & 1) ^ 1);
            mbar_arrive_expect_tx(bar_full + 8 * OB_RX, P::SZ_S);
            tma_load_5d_hint(sbase + P::OFF_X, &maps.s_c, bar_full + 8 * OB_RX, cx, y0, z0, tt, 0, pol_n);
            nX++;
        };
        auto load_sb = [&](int tt) {  // block B into the Y object's buffer
            mbar_wait(bar_empty + 8 * OB_RY, (nY & 1) ^ 1);
            mbar_arrive_expect_tx(bar_full + 8 * OB_RY, P::SZ_S);
            tma_load_5d_hint(sbase + P::OFF_Y, &maps.s_c, bar_full + 8 * OB_RY, cx, y0, z0, tt, 18, pol_n);
            nY++;
        };
        auto wrap = [&](int tt) { return (tt < 0) ? tt + T : (tt >= T) ? tt - T : tt; };

        const int t0 = it.t0, tc = prm.tchunk;
        // prologue: psi(t0-1) seeds the carried half-spinor; then everything step 1 needs, and psi(t0+1)
        // (in the order in which the last step and the epilogue of the previous item free the buffers)
        load_c(wrap(t0 - 1));
        load_z(t0);
        load_x(t0);
        load_y(t0);
        load_t(wrap(t0 - 1));
        load_c(t0);
        load_c(wrap(t0 + 1));  // first use: step 2, or the epilogue if tc == 1
        for (int j = 1; j <= tc; j++) {
            const int t = t0 + j - 1;  // < T: a chunk does not wrap
            load_t(t);                 // U_T(t): the T phase of step j+1 (or of the epilogue)
            if (CLOVER) {
                load_sa(t);
                load_sb(t);
            }
            if (j < tc) {
                load_z(t + 1);
                load_c(wrap(t + 2));   // step j+2, or the epilogue (j + 2 == tc + 1)
                load_x(t + 1);
                load_y(t + 1);
            }
        }
    }
}

// ---------------------------------------------------------------- the kernel
template <class P, bool OPEN>
__global__ void __launch_bounds__(P::NTHREADS, 1) k_tmq(const __grid_constant__ TmaMaps maps, const TmaParams prm) {
    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t sbase = smem_u32(smem);
    const uint32_t bar_full = sbase + P::OFF_BAR, bar_empty = bar_full + OB_COUNT * 8;
    const int tid = threadIdx.x;
    typedef cd C;
    constexpr int BZ = P::BZ, BY = P::BY, BX = P::BX, N = P::N, G = P::G, SPW = 32 / G;
    constexpr bool CLOVER = (P::SELF == SELF_CLOVER), BLK = P::BLK;

    if (tid == 0) {
        if (sbase & 127u) __trap();  // TMA destinations need 128-byte alignment
        for (int k = 0; k < OB_COUNT; k++) {
            mbar_init(bar_full + 8 * k, 1);       // the producer's arrive(.expect_tx)
            mbar_init(bar_empty + 8 * k, P::NW);  // one arrive per compute warp
        }
        mbar_fence_init();
    }
    __syncthreads();

    const int T = prm.n[0], Z = prm.n[1], Y = prm.n[2], X = prm.n[3];

    if (tid >= P::NC) {
        // ======================= producer warpgroup: one thread issues every TMA =======================
        reg_dec<40>();
        if (tid == P::NC) producer<P>(maps, prm, smem, sbase, bar_full, bar_empty);
        return;
    }
    reg_inc<232>();
    // ======================= consumers: one thread per (site of the tile, right-hand side of the unit) =======================
    const int lane = tid & 31;
    const int r = BLK ? lane % G : lane / SPW;                         // right-hand side within the unit
    const int sid = (tid >> 5) * SPW + (BLK ? lane / G : lane % SPW);  // site within the tile
    const int lx = sid % BX, ly = (sid / BX) % BY, lz = sid / (BX * BY);
    constexpr uint32_t E = P::E, NS = N * E;
    constexpr uint32_t EP = E * P::RBK, NSP = N * EP;  // psi boxes: bytes per site, component stride of the interior
    const uint32_t own = sid * E;                                       // links, S
    const uint32_t ownp = BLK ? sid * EP + r * E : own + r * 12 * NS;   // psi interior of right-hand side r
    // operand addresses (bytes from the start of shared memory; interior psi relative to the C buffer in use)
    const uint32_t fz = (ly * BX + lx) * E, fy = (lz * BX + lx) * E, fx = (lz * BY + ly) * E;
    const uint32_t fzp = (ly * BX + lx) * EP + (BLK ? r * E : r * 12 * P::FZ * E);
    const uint32_t fyp = (lz * BX + lx) * EP + (BLK ? r * E : r * 12 * P::FY * E);
    const uint32_t fxp = (lz * BY + ly) * EP + (BLK ? r * E : r * 12 * P::FX * E);
    const bool zf_in = lz < BZ - 1, zb_in = lz > 0, yf_in = ly < BY - 1, yb_in = ly > 0, xf_in = lx < BX - 1, xb_in = lx > 0;
    const uint32_t z_pf = zf_in ? P::OFF_C + ownp + P::FZ * EP : P::OFF_ZHI + fzp, z_pf_s = zf_in ? NSP : P::FZ * EP;
    const uint32_t z_pb = zb_in ? P::OFF_C + ownp - P::FZ * EP : P::OFF_ZLO + fzp, z_pb_s = zb_in ? NSP : P::FZ * EP;
    const uint32_t z_ub = zb_in ? P::OFF_Z + own - P::FZ * E : P::OFF_ZUF + fz, z_ub_s = zb_in ? NS : P::FZ * E;
    const uint32_t y_pf = yf_in ? P::OFF_C + ownp + BX * EP : P::OFF_YHI + fyp, y_pf_s = yf_in ? NSP : P::FY * EP;
    const uint32_t y_pb = yb_in ? P::OFF_C + ownp - BX * EP : P::OFF_YLO + fyp, y_pb_s = yb_in ? NSP : P::FY * EP;
    const uint32_t y_ub = yb_in ? P::OFF_Y + own - BX * E : P::OFF_YUF + fy, y_ub_s = yb_in ? NS : P::FY * E;
    const uint32_t x_pf = xf_in ? P::OFF_C + ownp + EP : P::OFF_XHI + fxp, x_pf_s = xf_in ? NSP : P::FX * EP;
    const uint32_t x_pb = xb_in ? P::OFF_C + ownp - EP : P::OFF_XLO + fxp, x_pb_s = xb_in ? NSP : P::FX * EP;
    const uint32_t x_ub = xb_in ? P::OFF_X + own - E : P::OFF_XUF + fx, x_ub_s = xb_in ? NS : P::FX * E;

    auto release = [&](int ob) {
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8 * ob);
    };

    const long long V = prm.Vs;  // component stride
    const long long strideT = (long long)Z * Y * X;
    uint32_t nC = 0, nT = 0, nX = 0, nY = 0, nZ = 0;  // fills consumed so far
    C hprev[6];   // rows 0,1 of (1 + gamma_T) psi(t-1)
    C outp[12];   // out(t-1) still missing its forward-T hop

    const volatile int *mail = reinterpret_cast<const volatile int *>(smem + P::OFF_MAIL);
    for (uint32_t seq = 0;; seq++) {
        const uint32_t slot = seq & 1, mpar = (seq >> 1) & 1;
        mbar_wait(bar_full + 8 * (OB_ITEM0 + slot), mpar);
        const int item = mail[slot];
        release(OB_ITEM0 + slot);
        if (item < 0) break;
        const Item it = decode_item<P>(prm, item);
        const long long site0 = ((long long)(it.z0 + lz) * Y + (it.y0 + ly)) * X + (it.x0 + lx);
        // blocked layout: unit u at u * 12 * Vs * G elements, element (c, site, r) at (c * Vs + site) * G + r; its units are
        // padded to G right-hand sides, so every thread stores.  Plain layout: the last unit may hold fewer than G right-hand
        // sides (its boxes reach past the last one and are zero-filled); those threads do not store.
        C *__restrict__ out = reinterpret_cast<C *>(prm.out) + (BLK ? (long long)it.rhs0 * 12 * V + r : (long long)(it.rhs0 + r) * 12 * V);
        const bool live = BLK || r < it.ng;
        // open boundaries of a domain-decomposed sub-lattice: hops that would cross them are left out
        const int open = OPEN ? prm.open_mask : 0;
        const bool zf_on = !((open & 2) && it.z0 + lz == Z - 1), zb_on = !((open & 2) && it.z0 + lz == 0);
        const bool yf_on = !((open & 4) && it.y0 + ly == Y - 1), yb_on = !((open & 4) && it.y0 + ly == 0);
        const bool xf_on = !((open & 8) && it.x0 + lx == X - 1), xb_on = !((open & 8) && it.x0 + lx == 0);
        int t = (it.t0 == 0) ? T - 1 : it.t0 - 1;
        {   // prologue: seed the carried half-spinor from psi(t0-1)
            const uint32_t b = nC & 1, cb = b * P::SZ_C;
            C p[12];
            mbar_wait(bar_full + 8 * (OB_C0 + b), (nC >> 1) & 1);
#pragma unroll
            for (int c = 0; c < 12; c++) p[c] = lds<C>(smem, P::OFF_C + cb + ownp + c * NSP);
            project<0, +1>(hprev, p);
            if ((open & 1) && it.t0 == 0) {
#pragma unroll
                for (int c = 0; c < 6; c++) hprev[c] = mk<C>(0, 0);
            }
            release(OB_C0 + b);
            nC++;
        }
        for (int j = 1; j <= prm.tchunk + 1; j++) {
            const int tprev = t;
            t = (t + 1 == T) ? 0 : t + 1;
            const uint32_t b = nC & 1, cb = b * P::SZ_C;  // the C buffer that holds psi(t)
            C p[12], acc[12];
            {   // T phase: finish out(t-1) with its forward hop, start out(t) with its backward hop
                C u[9];
                mbar_wait(bar_full + 8 * OB_T, nT & 1);
                mbar_wait(bar_full + 8 * (OB_C0 + b), (nC >> 1) & 1);
                load_link<9, C>(u, smem, P::OFF_T + own, NS);
#pragma unroll
                for (int c = 0; c < 12; c++) p[c] = lds<C>(smem, P::OFF_C + cb + ownp + c * NSP);
                if (j > 1) {  // out(t-1) = outp - 1/2 (1 - gamma_T) U_T(t-1) psi(t)
                    C hf[6], gf[6], o[12];
                    project<0, -1>(hf, p);
                    su3_mul<false>(gf, u, hf);
                    reconstruct_axpy<0, -1>(o, outp, ((open & 1) && tprev == T - 1) ? 0.0 : -0.5, gf);
                    const long long ip = (long long)tprev * strideT + site0;
#pragma unroll
                    for (int c = 0; c < 12; c++)
                        if (live) __stcs(out + ((long long)c * V + ip) * P::RBK, o[c]);
                }
                if (j == prm.tchunk + 1) {  // epilogue step: nothing else to do for slice t
                    release(OB_T);
                    release(OB_C0 + b);
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
            mbar_wait(bar_full + 8 * OB_RX, nX & 1);
            hop_pair_smem<3, 9, C>(acc, smem, P::OFF_X + own, NS, x_pf + (xf_in ? cb : 0), x_pf_s, x_ub, x_ub_s,
                                   x_pb + (xb_in ? cb : 0), x_pb_s, xf_on, xb_on);
            release(OB_RX);
            nX++;
            mbar_wait(bar_full + 8 * OB_RY, nY & 1);
            hop_pair_smem<2, 9, C>(acc, smem, P::OFF_Y + own, NS, y_pf + (yf_in ? cb : 0), y_pf_s, y_ub, y_ub_s,
                                   y_pb + (yb_in ? cb : 0), y_pb_s, yf_on, yb_on);
            release(OB_RY);
            nY++;
            mbar_wait(bar_full + 8 * OB_RZ, nZ & 1);
            hop_pair_smem<1, 9, C>(acc, smem, P::OFF_Z + own, NS, z_pf + (zf_in ? cb : 0), z_pf_s, z_ub, z_ub_s,
                                   z_pb + (zb_in ? cb : 0), z_pb_s, zf_on, zb_on);
            release(OB_RZ);
            nZ++;
            release(OB_C0 + b);  // psi(t) is done (own site: in p)
            nC++;
            // self-coupling (a5) and combination (a6); the store waits for the forward-T hop
            if (CLOVER) {
#pragma unroll
                for (int blk = 0; blk < 2; blk++) {
                    const uint32_t so = (blk == 0 ? P::OFF_X : P::OFF_Y) + own;
                    mbar_wait(bar_full + 8 * (blk == 0 ? OB_RX : OB_RY), (blk == 0 ? nX : nY) & 1);
                    double d[6];
                    C a[15], s[6];
#pragma unroll
                    for (int q = 0; q < 3; q++) {
                        const C dd = lds<C>(smem, so + q * NS);
                        d[2 * q] = dd.x;
                        d[2 * q + 1] = dd.y;
                    }
#pragma unroll
                    for (int k = 0; k < 15; k++) a[k] = lds<C>(smem, so + (3 + k) * NS);
                    release(blk == 0 ? OB_RX : OB_RY);
                    herm6_mul(s, d, a, p + 6 * blk);
#pragma unroll
                    for (int c = 0; c < 6; c++)
                        outp[6 * blk + c] = mk<C>(fma(-0.5, acc[6 * blk + c].x, s[c].x), fma(-0.5, acc[6 * blk + c].y, s[c].y));
                }
                nX++;
                nY++;
            } else if (P::SELF == SELF_MASS) {
#pragma unroll
                for (int c = 0; c < 12; c++)
                    outp[c] = mk<C>(fma(prm.mass, p[c].x, -0.5 * acc[c].x), fma(prm.mass, p[c].y, -0.5 * acc[c].y));
            } else {
#pragma unroll
                for (int c = 0; c < 12; c++) outp[c] = mk<C>(-0.5 * acc[c].x, -0.5 * acc[c].y);
            }
        }
    }
}

// ---------------------------------------------------------------- host side
template <int BZ, int BY, int BX, bool BLK, int SELF> static cudaError_t launch_self(const KParams &p, cudaStream_t st) {
    using P = Plan<BZ, BY, BX, SELF, BLK>;
    return p.open_mask ? launch_tma_kernel<P>(k_tmq<P, true>, p, st, /*ucomp*/ 9, /*scomp*/ 18, CHUNK_COST_MODEL, /*rb*/ 4)
                       : launch_tma_kernel<P>(k_tmq<P, false>, p, st, /*ucomp*/ 9, /*scomp*/ 18, CHUNK_COST_MODEL, /*rb*/ 4);
}
template <int BZ, int BY, int BX, bool BLK> static cudaError_t launch(const KParams &p, int self, cudaStream_t st) {
    if (p.esize != 16) return cudaErrorNotSupported;  // FP64 only (two-row storage is ignored: nine-entry links are read)
    if (self == SELF_CLOVER) return launch_self<BZ, BY, BX, BLK, SELF_CLOVER>(p, st);
    if (self == SELF_MASS) return launch_self<BZ, BY, BX, BLK, SELF_MASS>(p, st);
    return launch_self<BZ, BY, BX, BLK, SELF_NONE>(p, st);
}
}  // namespace tmq

cudaError_t launch_tmq_2x4x8(const KParams &p, int self, cudaStream_t st) { return tmq::launch<2, 4, 8, false>(p, self, st); }
// ... on the blocked multi-RHS layout (WD_OPT_RHS_BLOCK = 4): p.psi / p.out are double2 [unit][12][Vs][4]
cudaError_t launch_tmqb_2x4x8(const KParams &p, int self, cudaStream_t st) { return tmq::launch<2, 4, 8, true>(p, self, st); }
}  // namespace wd
