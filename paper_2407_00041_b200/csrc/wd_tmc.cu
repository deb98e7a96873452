// wd_tmc.cu — the multi-right-hand-side kernel ("tmc_*", step a8 of SURVEY.md §8(a)): every thread applies
// the operator to TWO right-hand sides of its site, with each link and each block of S held in registers
// for both of them.
//
// The paper's observation: with several "tuples" the same link serves each of them.
// What round 1 measured (profiles/r1c §C6): the kernels that stage EVERY operand through shared memory
// (wd_tma.cu, wd_tmb.cu) converge to 4.4-5.0 G site·RHS/s once HBM is out of the way, because each site and
// right-hand side costs ~225 LDS.128 (3.6 KB) plus 0.9-1.7 KB of TMA writes on a 128 B/clk/SM pipe.  Sharing
// U and S between thread groups in shared memory (round 1's tmr kernels) changed the HBM/L2 bytes but not
// the LDS count, and was not faster.  Here the bytes that cross the shared-memory pipe are cut instead:
//   * psi (interior, double-buffered, and the six spatial faces) of G = 2 right-hand sides comes in by TMA,
//     as in wd_tmb.cu — this is the only data with reuse across threads (each psi serves 9 sites);
//   * U and S are read by every thread for its own site with LDG.128 straight into registers (coalesced:
//     the device layout is SoA over sites), nine complex numbers at a time through two alternating register
//     buffers, the next nine in flight while the current nine are used for BOTH right-hand sides.  The
//     backward link U_mu(x-mu) is the neighbour site's own link: an L1 hit for most of the tile.  One chunk of
//     lookahead covers an L2 hit, not an HBM miss (first version: 35 ms on cfg 5, every chunk a dependent HBM round
//     trip), so the producer thread warms L2 one T slice ahead with eleven cp.async.bulk.prefetch.tensor boxes per
//     step (4 links, 3 face links, 4 quarter-blocks of S): bytes in flight without registers or shared memory;
//   * per site and right-hand side: 108 LDS.128 + 504 B of TMA writes (2.2 KB) + 50 LDG.128 (0.8 KB)
//     instead of 5.3 KB, and two independent dependency chains per thread for the 8.4-cycle DFMA latency.
// With several units of two right-hand sides per tile (item order of wd_tma_common.cuh) U and S come from
// HBM once and from L2 for the other units.  T direction as in wd_tmb.cu: acc[G][12] is the only state carried
// from phase to phase; at the end of step t the forward hop completes out(t) and the backward hop of slice
// t+1 starts the next accumulator, both with U_T(t) in registers.
#include <cstdio>
#include <cstdlib>
#include <type_traits>

#include "wd_tma_common.cuh"
#include "wd_smem_ops.cuh"

namespace wd {
namespace tmc {

// ---------------------------------------------------------------- shared-memory plan
//   C   psi_g(t) interior [G][12][N], TWO buffers (fill n in buffer n & 1)
//   PZ  psi_g faces z0-1 | z0+BZ  [G][2][12][FZ];  PY, PX alike
enum { OB_C = 0, OB_C1, OB_PZ, OB_PY, OB_PX, OB_ITEM0, OB_ITEM1, OB_COUNT };

template <int BZ_, int BY_, int BX_, int SELF_> struct Plan {
    static constexpr int BZ = BZ_, BY = BY_, BX = BX_, SELF = SELF_;
    static constexpr int G = 2;              // right-hand sides per work item = per thread
    static constexpr int N = BZ * BY * BX;   // sites per tile = compute threads
    static constexpr int CTAS_PER_SM = 1;
    static constexpr int XW = 1;             // sites per row of an X-face box (wd_tma.cu: 2 for 8-byte elements)
    static constexpr int NW = N / 32;
    static constexpr int NTHREADS = N + 32;  // + the producer warp
    static constexpr int FZ = BY * BX, FY = BZ * BX, FX = BZ * BY;
    static constexpr uint32_t E = 16;
    static constexpr uint32_t SZ_C1 = 12 * N * E, SZ_C = G * SZ_C1;  // one right-hand side; one buffer
    static constexpr uint32_t OFF_C = 0;
    static constexpr uint32_t SZ_FZ = 12 * FZ * E, SZ_FY = 12 * FY * E, SZ_FX = 12 * FX * E;  // one face of one RHS
    static constexpr uint32_t OFF_PZ = OFF_C + 2 * SZ_C, SZ_PZ = G * 2 * SZ_FZ;
    static constexpr uint32_t OFF_PY = OFF_PZ + SZ_PZ, SZ_PY = G * 2 * SZ_FY;
    static constexpr uint32_t OFF_PX = OFF_PY + SZ_PY, SZ_PX = G * 2 * SZ_FX;
    static constexpr uint32_t OFF_BAR = OFF_PX + SZ_PX;
    static constexpr uint32_t OFF_MAIL = OFF_BAR + 2 * OB_COUNT * 8;
    static constexpr uint32_t SMEM = OFF_MAIL + 16;
    static_assert(N % 32 == 0 && FZ % 8 == 0 && FY % 8 == 0 && FX % 8 == 0, "tile faces must keep 128-byte alignment");
    static_assert(SMEM <= 232448, "shared-memory plan exceeds 227 KB");
};

// nine complex numbers of a device-layout field (component stride Vs) for one site, read-only path
__device__ __forceinline__ void ldg9(cd a[9], const cd *__restrict__ base, long long Vs) {
#pragma unroll
    for (int k = 0; k < 9; k++) a[k] = __ldg(base + (long long)k * Vs);
}

// the same nine into L1 without a destination register (two chunks ahead of their use)
__device__ __forceinline__ void pf9(const cd *__restrict__ base, long long Vs) {
#pragma unroll
    for (int k = 0; k < 9; k++) asm volatile("prefetch.global.L1 [%0];" ::"l"(base + (long long)k * Vs));
}

// ---------------------------------------------------------------- the kernel
template <class P>
__global__ void __launch_bounds__(P::NTHREADS, 1) k_tmc(const __grid_constant__ TmaMaps maps, const TmaParams prm) {
    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t sbase = smem_u32(smem);
    const uint32_t bar_full = sbase + P::OFF_BAR, bar_empty = bar_full + OB_COUNT * 8;
    const int tid = threadIdx.x;
    constexpr int BZ = P::BZ, BY = P::BY, BX = P::BX, N = P::N, G = P::G;
    constexpr bool CLOVER = (P::SELF == SELF_CLOVER);

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

    if (tid >= N) {
        // ======================= producer: one thread issues every TMA =======================
        // Per item: psi(t0), then per step the faces of slice t (in the order the consumers release them) and
        // psi(t+1) into the other C buffer.  Every wait is for a buffer the consumers release in this same order.
        if (tid != N) return;
        tma_prefetch_desc(&maps.psi_c); tma_prefetch_desc(&maps.psi_z); tma_prefetch_desc(&maps.psi_y);
        tma_prefetch_desc(&maps.psi_x); tma_prefetch_desc(&maps.u_c);   tma_prefetch_desc(&maps.u_z);
        tma_prefetch_desc(&maps.u_y);   tma_prefetch_desc(&maps.u_x);   tma_prefetch_desc(&maps.s_c);
        const uint64_t pol_p = l2_policy_evict_normal();
        uint32_t nC = 0, nF = 0;
        // U and S of slice tt into L2: what the consumers' LDGs of that slice will hit
        auto warm_l2 = [&](int cx, int y0, int z0, int zlo, int ylo, int cxlo, int tt) {
#pragma unroll
            for (int mu = 0; mu < 4; mu++) tma_prefetch_5d(&maps.u_c, cx, y0, z0, tt, 9 * mu);
            tma_prefetch_5d(&maps.u_z, cx, y0, zlo, tt, 9);
            tma_prefetch_5d(&maps.u_y, cx, ylo, z0, tt, 18);
            tma_prefetch_5d(&maps.u_x, cxlo, y0, z0, tt, 27);
            if (CLOVER) {
#pragma unroll
                for (int q = 0; q < 4; q++) tma_prefetch_5d(&maps.s_c, cx, y0, z0, tt, 9 * q);
            }
        };
        volatile int *mail = reinterpret_cast<volatile int *>(smem + P::OFF_MAIL);
        auto load_c = [&](int cx, int y0, int z0, int tt, const int pc[G]) {
            const uint32_t b = nC & 1, ob = OB_C + b;
            mbar_wait(bar_empty + 8 * ob, ((nC >> 1) & 1) ^ 1);
            mbar_arrive_expect_tx(bar_full + 8 * ob, P::SZ_C);
#pragma unroll
            for (int g = 0; g < G; g++)
                tma_load_5d_hint(sbase + P::OFF_C + b * P::SZ_C + g * P::SZ_C1, &maps.psi_c, bar_full + 8 * ob, cx, y0, z0, tt,
                                 pc[g], pol_p);
            nC++;
        };
        for (uint32_t seq = 0;; seq++) {
            const int item = fetch_item(prm, seq);
            const uint32_t slot = seq & 1, mpar = (seq >> 1) & 1;
            mbar_wait(bar_empty + 8 * (OB_ITEM0 + slot), mpar ^ 1);
            mail[slot] = item;
            mbar_arrive(bar_full + 8 * (OB_ITEM0 + slot));
            if (item < 0) break;
            const Item it = decode_item<P>(prm, item);
            const int cx = 2 * it.x0, y0 = it.y0, z0 = it.z0;  // dim-0 coordinates count doubles
            int pc[G];  // first component of each right-hand side; a unit with one RHS loads it twice
#pragma unroll
            for (int g = 0; g < G; g++) pc[g] = 12 * (it.rhs0 + ((g < it.ng) ? g : 0));
            const int zlo = (z0 == 0) ? Z - 1 : z0 - 1, zhi = (z0 + BZ == Z) ? 0 : z0 + BZ;
            const int ylo = (y0 == 0) ? Y - 1 : y0 - 1, yhi = (y0 + BY == Y) ? 0 : y0 + BY;
            const int cxlo = 2 * ((it.x0 == 0) ? X - 1 : it.x0 - 1), cxhi = 2 * ((it.x0 + BX == X) ? 0 : it.x0 + BX);
            int t = it.t0;
            warm_l2(cx, y0, z0, zlo, ylo, cxlo, t);
            load_c(cx, y0, z0, t, pc);
            for (int j = 1; j <= prm.tchunk; j++) {
                if (j < prm.tchunk) warm_l2(cx, y0, z0, zlo, ylo, cxlo, (t + 1 == T) ? 0 : t + 1);
                const uint32_t pe = (nF & 1) ^ 1;
                mbar_wait(bar_empty + 8 * OB_PZ, pe);
                mbar_arrive_expect_tx(bar_full + 8 * OB_PZ, P::SZ_PZ);
#pragma unroll
                for (int g = 0; g < G; g++) {
                    const uint32_t d = sbase + P::OFF_PZ + g * 2 * P::SZ_FZ;
                    tma_load_5d_hint(d, &maps.psi_z, bar_full + 8 * OB_PZ, cx, y0, zlo, t, pc[g], pol_p);
                    tma_load_5d_hint(d + P::SZ_FZ, &maps.psi_z, bar_full + 8 * OB_PZ, cx, y0, zhi, t, pc[g], pol_p);
                }
                mbar_wait(bar_empty + 8 * OB_PY, pe);
                mbar_arrive_expect_tx(bar_full + 8 * OB_PY, P::SZ_PY);
#pragma unroll
                for (int g = 0; g < G; g++) {
                    const uint32_t d = sbase + P::OFF_PY + g * 2 * P::SZ_FY;
                    tma_load_5d_hint(d, &maps.psi_y, bar_full + 8 * OB_PY, cx, ylo, z0, t, pc[g], pol_p);
                    tma_load_5d_hint(d + P::SZ_FY, &maps.psi_y, bar_full + 8 * OB_PY, cx, yhi, z0, t, pc[g], pol_p);
                }
                mbar_wait(bar_empty + 8 * OB_PX, pe);
                mbar_arrive_expect_tx(bar_full + 8 * OB_PX, P::SZ_PX);
#pragma unroll
                for (int g = 0; g < G; g++) {
                    const uint32_t d = sbase + P::OFF_PX + g * 2 * P::SZ_FX;
                    tma_load_5d_hint(d, &maps.psi_x, bar_full + 8 * OB_PX, cxlo, y0, z0, t, pc[g], pol_p);
                    tma_load_5d_hint(d + P::SZ_FX, &maps.psi_x, bar_full + 8 * OB_PX, cxhi, y0, z0, t, pc[g], pol_p);
                }
                nF++;
                t = (t + 1 == T) ? 0 : t + 1;
                load_c(cx, y0, z0, t, pc);  // psi(t+1): forward-T hop of this slice, centre of the next step
            }
        }
        return;
    }
    // ======================= consumers: thread = site, G right-hand sides each =======================
    const int lane = tid & 31;
    const int lx = tid % BX, ly = (tid / BX) % BY, lz = tid / (BX * BY);
    constexpr uint32_t E = P::E, NS = N * E;
    const uint32_t own = tid * E;
    // psi operand addresses of right-hand side 0 (bytes from the start of shared memory): interior (relative to
    // the C buffer in use) or face storage; (second right-hand side: + z_pf_g etc.)
    const uint32_t fz = (ly * BX + lx) * E, fy = (lz * BX + lx) * E, fx = (lz * BY + ly) * E;
    const bool zf_in = lz < BZ - 1, zb_in = lz > 0, yf_in = ly < BY - 1, yb_in = ly > 0, xf_in = lx < BX - 1, xb_in = lx > 0;
    const uint32_t z_pf = zf_in ? P::OFF_C + own + P::FZ * E : P::OFF_PZ + P::SZ_FZ + fz, z_pf_s = zf_in ? NS : P::FZ * E;
    const uint32_t z_pb = zb_in ? P::OFF_C + own - P::FZ * E : P::OFF_PZ + fz, z_pb_s = zb_in ? NS : P::FZ * E;
    const uint32_t y_pf = yf_in ? P::OFF_C + own + BX * E : P::OFF_PY + P::SZ_FY + fy, y_pf_s = yf_in ? NS : P::FY * E;
    const uint32_t y_pb = yb_in ? P::OFF_C + own - BX * E : P::OFF_PY + fy, y_pb_s = yb_in ? NS : P::FY * E;
    const uint32_t x_pf = xf_in ? P::OFF_C + own + E : P::OFF_PX + P::SZ_FX + fx, x_pf_s = xf_in ? NS : P::FX * E;
    const uint32_t x_pb = xb_in ? P::OFF_C + own - E : P::OFF_PX + fx, x_pb_s = xb_in ? NS : P::FX * E;
    // distance between the two right-hand sides of an operand: interior SZ_C1, faces 2 * (one face)
    const uint32_t z_pf_g = zf_in ? P::SZ_C1 : 2 * P::SZ_FZ, z_pb_g = zb_in ? P::SZ_C1 : 2 * P::SZ_FZ;
    const uint32_t y_pf_g = yf_in ? P::SZ_C1 : 2 * P::SZ_FY, y_pb_g = yb_in ? P::SZ_C1 : 2 * P::SZ_FY;
    const uint32_t x_pf_g = xf_in ? P::SZ_C1 : 2 * P::SZ_FX, x_pb_g = xb_in ? P::SZ_C1 : 2 * P::SZ_FX;

    auto release = [&](int ob) {
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8 * ob);
    };
    auto wait_full = [&](int ob, uint32_t parity) { mbar_wait(bar_full + 8 * ob, parity); };

    const long long Vs = prm.Vs;
    const long long strideY = X, strideZ = (long long)Y * X, strideT = (long long)Z * Y * X;
    const cd *__restrict__ U = prm.U;
    const cd *__restrict__ S = prm.S;
    uint32_t nC = 0, nF = 0;
    cd acc[G][12];
    cd ua[9], ub[9];  // the two alternating register buffers of the U / S stream

    // both hops' arithmetic for the G right-hand sides with one link in registers
    auto hops = [&](auto mu_tag, auto sign_tag, const cd u[9], uint32_t p, uint32_t stride, uint32_t gstep) {
        constexpr int MU = decltype(mu_tag)::value, SIGN = decltype(sign_tag)::value;
#pragma unroll
        for (int g = 0; g < G; g++) {
            hop_row_smem<MU, SIGN, 0>(acc[g], smem, p + g * gstep, stride, u);
            hop_row_smem<MU, SIGN, 1>(acc[g], smem, p + g * gstep, stride, u);
        }
    };
    // half of a 6x6 block of S in registers: acc_g[6b..6b+5] += (part of B_b) (-2 psi_g)
    auto s_chunk = [&](auto h_tag, const cd a[9], uint32_t cb, int b) {
        constexpr int H = decltype(h_tag)::value;
#pragma unroll
        for (int g = 0; g < G; g++) {
            cd q[6];
#pragma unroll
            for (int c = 0; c < 6; c++) {
                const cd v = lds(smem, P::OFF_C + cb + g * P::SZ_C1 + own + (6 * b + c) * NS);
                q[c] = make_double2(-2.0 * v.x, -2.0 * v.y);
            }
            herm6_half_add_reg<H>(acc[g] + 6 * b, a, q);
        }
    };
    using I0 = std::integral_constant<int, 0>;
    using I1 = std::integral_constant<int, 1>;
    using I2 = std::integral_constant<int, 2>;
    using I3 = std::integral_constant<int, 3>;
    using FWD = std::integral_constant<int, -1>;
    using BWD = std::integral_constant<int, +1>;

    const volatile int *mail = reinterpret_cast<const volatile int *>(smem + P::OFF_MAIL);
    for (uint32_t seq = 0;; seq++) {
        const uint32_t mslot = seq & 1, mpar = (seq >> 1) & 1;
        wait_full(OB_ITEM0 + mslot, mpar);
        const int item = mail[mslot];
        release(OB_ITEM0 + mslot);
        if (item < 0) break;
        const Item it = decode_item<P>(prm, item);
        const int z = it.z0 + lz, y = it.y0 + ly, x = it.x0 + lx;
        const long long site0 = ((long long)z * Y + y) * X + x;
        // site-index offsets of the backward neighbours (periodic wrap, a1)
        const long long dzb = (z == 0) ? (long long)(Z - 1) * strideZ : -strideZ;
        const long long dyb = (y == 0) ? (long long)(Y - 1) * strideY : -strideY;
        const long long dxb = (x == 0) ? (long long)(X - 1) : -1;
        int t = it.t0;
        {   // prologue: acc_g = backward-T hop of slice t0, (1 + gamma_T) U_T(t0-1)^H psi_g(t0-1), operands by LDG
            const int tm = (t == 0) ? T - 1 : t - 1;
            const long long im = (long long)tm * strideT + site0;
            ldg9(ua, U + im, Vs);
#pragma unroll
            for (int g = 0; g < G; g++) {
                const cd *__restrict__ pg = prm.psi + (long long)(it.rhs0 + ((g < it.ng) ? g : 0)) * 12 * Vs + im;
#pragma unroll
                for (int c = 0; c < 12; c++) acc[g][c] = make_double2(0.0, 0.0);
                hop_row_ldg<0, +1, 0>(acc[g], pg, Vs, ua);
                hop_row_ldg<0, +1, 1>(acc[g], pg, Vs, ua);
            }
            ldg9(ua, U + 9 * Vs + (long long)t * strideT + site0, Vs);  // U_Z(x) of the first slice
        }
        for (int j = 1; j <= prm.tchunk; j++) {
            const bool last = (j == prm.tchunk);
            const uint32_t cb = (nC & 1) ? P::SZ_C : 0;  // C buffer holding psi(t)
            if (j == 1) wait_full(OB_C + (nC & 1), (nC >> 1) & 1);
            const uint32_t pf = nF & 1;
            const long long i = (long long)t * strideT + site0;
            // The U / S stream of a step, nine complex numbers per chunk:
            //   U_Z(x) U_Z(x-z) U_Y(x) U_Y(x-y) [S0 S1 S2 S3] U_X(x) U_X(x-x) U_T(x) | U_Z(x) of the next slice ...
            // chunk k is used from registers while chunk k+1 is in flight to the other register buffer (ldg9) and
            // chunk k+2 is on its way into L1 (pf9).
            const cd *__restrict__ Ui = U + i;
            const cd *__restrict__ Si = S + i;
            // ---- Z: ua = U_Z(x)
            wait_full(OB_PZ, pf);
            ldg9(ub, Ui + 9 * Vs + dzb, Vs);
            pf9(Ui + 18 * Vs, Vs);
            hops(I1{}, FWD{}, ua, z_pf + (zf_in ? cb : 0), z_pf_s, z_pf_g);
            ldg9(ua, Ui + 18 * Vs, Vs);
            pf9(Ui + 18 * Vs + dyb, Vs);
            hops(I1{}, BWD{}, ub, z_pb + (zb_in ? cb : 0), z_pb_s, z_pb_g);
            release(OB_PZ);
            // ---- Y: ua = U_Y(x)
            wait_full(OB_PY, pf);
            ldg9(ub, Ui + 18 * Vs + dyb, Vs);
            if (CLOVER) pf9(Si, Vs);
            else pf9(Ui + 27 * Vs, Vs);
            hops(I2{}, FWD{}, ua, y_pf + (yf_in ? cb : 0), y_pf_s, y_pf_g);
            if (CLOVER) {
                ldg9(ua, Si, Vs);
                pf9(Si + 9 * Vs, Vs);
            } else {
                ldg9(ua, Ui + 27 * Vs, Vs);
                pf9(Ui + 27 * Vs + dxb, Vs);
            }
            hops(I2{}, BWD{}, ub, y_pb + (yb_in ? cb : 0), y_pb_s, y_pb_g);
            release(OB_PY);
            if (CLOVER) {  // ---- S: four chunks of nine slots (block A: 0..8, 9..17; block B: 18..26, 27..35)
                ldg9(ub, Si + 9 * Vs, Vs);
                pf9(Si + 18 * Vs, Vs);
                s_chunk(I0{}, ua, cb, 0);
                ldg9(ua, Si + 18 * Vs, Vs);
                pf9(Si + 27 * Vs, Vs);
                s_chunk(I1{}, ub, cb, 0);
                ldg9(ub, Si + 27 * Vs, Vs);
                pf9(Ui + 27 * Vs, Vs);
                s_chunk(I0{}, ua, cb, 1);
                ldg9(ua, Ui + 27 * Vs, Vs);
                pf9(Ui + 27 * Vs + dxb, Vs);
                s_chunk(I1{}, ub, cb, 1);
            }
            // ---- X: ua = U_X(x)
            wait_full(OB_PX, pf);
            ldg9(ub, Ui + 27 * Vs + dxb, Vs);
            pf9(Ui, Vs);
            hops(I3{}, FWD{}, ua, x_pf + (xf_in ? cb : 0), x_pf_s, x_pf_g);
            ldg9(ua, Ui, Vs);  // U_T(x, t)
            if (!last) pf9(Ui + strideT + 9 * Vs - ((t + 1 == T) ? (long long)T * strideT : 0), Vs);
            hops(I3{}, BWD{}, ub, x_pb + (xb_in ? cb : 0), x_pb_s, x_pb_g);
            release(OB_PX);
            nF++;
            {   // ---- T: forward hop (1 - gamma_T) U_T(t) psi(t+1) completes out(t); the backward hop of slice t+1,
                // (1 + gamma_T) U_T(t)^H psi(t), starts the next accumulator.  ua = U_T(x, t).
                const uint32_t cn = cb ^ P::SZ_C;  // psi(t+1) is in the other C buffer
                const int tn = (t + 1 == T) ? 0 : t + 1;
                wait_full(OB_C + ((nC + 1) & 1), ((nC + 1) >> 1) & 1);
                if (!last) {
                    const cd *__restrict__ Un = U + (long long)tn * strideT + site0;
                    ldg9(ub, Un + 9 * Vs, Vs);  // U_Z(x) of the next slice
                    pf9(Un + 9 * Vs + dzb, Vs);
                }
                hops(I0{}, FWD{}, ua, P::OFF_C + cn + own, NS, P::SZ_C1);
#pragma unroll
                for (int g = 0; g < G; g++) {
                    const uint32_t pown = P::OFF_C + cb + g * P::SZ_C1 + own;  // psi_g(t) of the own site
                    if (g < it.ng) {
                        cd *__restrict__ out = reinterpret_cast<cd *>(prm.out) + (long long)(it.rhs0 + g) * 12 * Vs + i;
#pragma unroll
                        for (int c = 0; c < 12; c++) {
                            cd o = make_double2(-0.5 * acc[g][c].x, -0.5 * acc[g][c].y);
                            if (P::SELF == SELF_MASS) {
                                const cd q = lds(smem, pown + c * NS);
                                o = make_double2(fma(prm.mass, q.x, o.x), fma(prm.mass, q.y, o.y));
                            }
                            __stcs(out + (long long)c * Vs, o);
                        }
                    }
                    if (!last) {
#pragma unroll
                        for (int c = 0; c < 12; c++) acc[g][c] = make_double2(0.0, 0.0);
                        hop_row_smem<0, +1, 0>(acc[g], smem, pown, NS, ua);
                        hop_row_smem<0, +1, 1>(acc[g], smem, pown, NS, ua);
                    }
                }
                release(OB_C + (nC & 1));  // psi(t) is done; psi(t+1) stays for the next step
                nC++;
                if (last) {                // ... unless this was the item's last slice
                    release(OB_C + (nC & 1));
                    nC++;
                }
#pragma unroll
                for (int k = 0; k < 9; k++) ua[k] = ub[k];
                t = tn;
            }
        }
    }
}

// ---------------------------------------------------------------- host side
template <int BZ, int BY, int BX, int SELF> static cudaError_t launch_self(const KParams &p, cudaStream_t st) {
    using P = Plan<BZ, BY, BX, SELF>;
    if (p.open_mask) return cudaErrorNotSupported;  // sub-lattices of a domain decomposition: wd_tma.cu / wd_tmb.cu
    // units of two right-hand sides that share a tile's U and S through L2: three (six right-hand sides in flight per tile)
    return launch_tma_kernel<P>(k_tmc<P>, p, st, /*ucomp*/ 9, /*scomp*/ 9, CHUNK_SHORT, /*rb*/ 3);
}

template <int BZ, int BY, int BX> static cudaError_t launch(const KParams &p, int self, cudaStream_t st) {
    if (self == SELF_CLOVER) return launch_self<BZ, BY, BX, SELF_CLOVER>(p, st);
    if (self == SELF_MASS) return launch_self<BZ, BY, BX, SELF_MASS>(p, st);
    return launch_self<BZ, BY, BX, SELF_NONE>(p, st);
}
}  // namespace tmc

cudaError_t launch_tmc_2x4x16(const KParams &p, int self, cudaStream_t st) { return tmc::launch<2, 4, 16>(p, self, st); }
}  // namespace wd
