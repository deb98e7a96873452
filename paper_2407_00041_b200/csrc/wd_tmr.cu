// wd_tmr.cu — the multi-right-hand-side TMA kernel ("tmr_*", step a8 of SURVEY.md §8(a)): G groups of
// compute threads apply the operator to G right-hand sides of ONE tile at the same time and share the
// links and S of that tile in shared memory.
//
// The paper's observation: with several "tuples" the same link is used for each of
// them.  wd_tma.cu / wd_tmb.cu share U and S between right-hand sides only through L2 (each CTA still pulls
// them into its own shared memory), and their one compute warp per SM sub-partition is what bounds a
// multi-RHS application (profiles/r1c: 3.7 us per 128-site tile step, IPC 0.25).  Here:
//   * the tile has 64 sites (2x4x8); a compute group is 64 threads = 2 warps, one thread per site;
//   * G = 3 groups work on 3 right-hand sides: 6 compute warps + the producer warp = 224 threads, which
//     still leaves 255 registers per thread (a 4th group would cap them at 168);
//   * U_Z/U_Y/U_X (interior + face), S and U_T are loaded ONCE per tile step and read by all groups: per
//     site and RHS HBM/L2 supply 384 + 1152/G bytes;
//   * psi and its six faces are per group (two psi buffers each), with their own mbarriers, so the groups
//     drift freely inside a step and hide each other's latencies.
// Everything else is wd_tmb.cu's scheme: psi double-buffered, acc[12] the only state carried between phases,
// S folded in as -2 S psi, forward-T hop and store at the end of the step, producer = resumable state machine,
// atomic work queue.
#include <cstdio>
#include <cstdlib>
#include <vector>

#include "wd_internal.h"
#include "wd_math.cuh"
#include "wd_tma.cuh"
#include "wd_smem_ops.cuh"

namespace wd {
namespace tmr {

// ---------------------------------------------------------------- shared-memory plan
// shared objects:  UZ = U_Z(t) interior [9][N] | face z0-1 [9][FZ];  UY, UX alike;
//                  R  = ring of kRing [9][N] slots: S1, S2 (block A), S3, S4 (block B), T = U_T(t)
// per group g:     C  = psi_g(t) interior [12][N], two buffers;  PZ = psi_g faces z0-1 | z0+BZ [12][FZ] each;  PY, PX
constexpr int kRing = 6;  // ring slots: all groups must be done with a slot before it is refilled, so the ring is
                          // what couples the groups; six slots for five objects per step let them drift by a step
enum { OB_UZ = 0, OB_UY, OB_UX, OB_R, OB_ITEM0 = OB_R + kRing, OB_ITEM1, OB_GROUP };  // then 5 per group:
enum { GB_C = 0, GB_C1, GB_PZ, GB_PY, GB_PX, GB_COUNT };

template <int BZ_, int BY_, int BX_, int SELF_, int G_> struct Plan {
    static constexpr int BZ = BZ_, BY = BY_, BX = BX_, SELF = SELF_, G = G_;
    static constexpr int N = BZ * BY * BX;       // sites per tile = threads per compute group
    static constexpr int NW = N / 32;            // warps per group
    static constexpr int NTHREADS = G * N + 32;  // + the producer warp
    static constexpr int FZ = BY * BX, FY = BZ * BX, FX = BZ * BY;  // sites per face
    static constexpr uint32_t E = 16;
    static constexpr uint32_t SZ_C = 12 * N * E, SZ_U = 9 * N * E;
    static constexpr uint32_t OFF_UZ = 0, OFF_UZF = OFF_UZ + SZ_U, SZ_UZ = SZ_U + 9 * FZ * E;
    static constexpr uint32_t OFF_UY = OFF_UZ + SZ_UZ, OFF_UYF = OFF_UY + SZ_U, SZ_UY = SZ_U + 9 * FY * E;
    static constexpr uint32_t OFF_UX = OFF_UY + SZ_UY, OFF_UXF = OFF_UX + SZ_U, SZ_UX = SZ_U + 9 * FX * E;
    static constexpr uint32_t OFF_R = OFF_UX + SZ_UX;
    static constexpr uint32_t OFF_G = OFF_R + kRing * SZ_U;  // group regions start here
    // offsets inside a group region
    static constexpr uint32_t GO_C = 0;
    static constexpr uint32_t GO_ZLO = GO_C + 2 * SZ_C, GO_ZHI = GO_ZLO + 12 * FZ * E, SZ_PZ = 24 * FZ * E;
    static constexpr uint32_t GO_YLO = GO_ZHI + 12 * FZ * E, GO_YHI = GO_YLO + 12 * FY * E, SZ_PY = 24 * FY * E;
    static constexpr uint32_t GO_XLO = GO_YHI + 12 * FY * E, GO_XHI = GO_XLO + 12 * FX * E, SZ_PX = 24 * FX * E;
    static constexpr uint32_t SZ_G = GO_XHI + 12 * FX * E;
    static constexpr uint32_t OFF_BAR = OFF_G + G * SZ_G;
    static constexpr int NBAR = OB_GROUP + G * GB_COUNT;
    static constexpr uint32_t OFF_MAIL = OFF_BAR + 2 * NBAR * 8;  // int[2][2]: (item, number of active groups) per slot
    static constexpr uint32_t SMEM = OFF_MAIL + 16;
    static_assert(N % 32 == 0 && FZ % 8 == 0 && FY % 8 == 0 && FX % 8 == 0, "tile faces must keep 128-byte alignment");
    static_assert(SMEM <= 232448, "shared-memory plan exceeds 227 KB");
};

struct TmaMaps {
    CUtensorMap psi_c, psi_z, psi_y, psi_x;  // boxes: interior, z-face, y-face, x-face (12 components)
    CUtensorMap u_c, u_z, u_y, u_x;          // same shapes, 9 components (one link)
    CUtensorMap s_c;                         // interior box, 9 components (half of a 6x6 block)
};

struct TmaParams {
    double2 *out;
    long long V, Vs;     // sites, component stride
    int n[4];
    int ntx, nty, ntz;   // tiles per direction
    int py, pz;          // rasterisation panel (in tiles); py | nty, pz | ntz
    int tchunk, ntc;     // T steps per work item, items per tile
    int nrhs, nblk;      // right-hand sides in this launch; blocks of up to G of them
    int nitems;          // ntx*nty*ntz*ntc*nblk
    double mass;
    int flags;           // WD_TMA_FLAGS (experiments; 0 = production): 1 S evict_normal, 2 U evict_first, 4 psi evict_last,
                         // 16 static round-robin items
    unsigned int *sched; // [0] next item, [1] CTAs finished
};

struct Item {
    int x0, y0, z0, t0, rhs0, ng;  // first right-hand side of the block, number of active groups
};

// Item order (slowest to fastest): T chunk, block of right-hand sides, tile (panel order).
template <class P> __device__ __forceinline__ Item decode_item(const TmaParams &prm, int item) {
    const int ntiles = prm.ntx * prm.nty * prm.ntz;
    const int per_chunk = ntiles * prm.nblk;
    const int chunk = item / per_chunk;
    int rem = item - chunk * per_chunk;
    const int blk = rem / ntiles;
    const int tile = rem - blk * ntiles;
    const int tpp = prm.ntx * prm.py * prm.pz;  // tiles per rasterisation panel
    const int panel = tile / tpp;
    int r = tile - panel * tpp;
    const int tx = r % prm.ntx;
    r /= prm.ntx;
    const int tyi = r % prm.py, tzi = r / prm.py;
    const int npy = prm.nty / prm.py;
    Item it;
    it.x0 = tx * P::BX;
    it.y0 = ((panel % npy) * prm.py + tyi) * P::BY;
    it.z0 = ((panel / npy) * prm.pz + tzi) * P::BZ;
    it.t0 = chunk * prm.tchunk;
    it.rhs0 = blk * P::G;
    it.ng = min(P::G, prm.nrhs - it.rhs0);
    return it;
}

// ---------------------------------------------------------------- the producer (one thread)
// Resumable state machine (see wd_tmb.cu).  Sequence per work item, g running over all G groups:
//   [fetch item] [psi_g(t0-1)]* [U_T(t0-1)] [psi_g(t0)]*   then per step t:
//   [UZ] [PZ_g]* [UY] [PY_g]* [S1] [S2] [S3] [S4] [UX] [PX_g]* [psi_g(t+1)]* [U_T(t)]
// A group without a right-hand side of its own (last block when nrhs % G != 0) is fed the block's first
// right-hand side and goes through the barrier protocol without computing or storing.
enum { ST_FETCH = 0, ST_PRO_C, ST_PRO_T, ST_PRO_C2, ST_UZ, ST_PZ, ST_UY, ST_PY, ST_S1, ST_S2, ST_S3, ST_S4, ST_UX, ST_PX, ST_C, ST_T };

template <class P> struct Producer {
    uint32_t nC, nR, nF, seq;  // fills issued so far: C buffers (per group), ring slots, per-step objects; items fetched
    int stage, g, j, t;        // g = group whose object is next; j = step within the item, t = its T slice
    int cx, y0, z0, rhs0, ng, zlo, zhi, ylo, yhi, cxlo, cxhi;
    bool done;
    uint64_t pol_n, pol_s, pol_u, pol_p;

    __device__ __forceinline__ void init(const TmaMaps &maps, const TmaParams &prm) {
        tma_prefetch_desc(&maps.psi_c); tma_prefetch_desc(&maps.psi_z); tma_prefetch_desc(&maps.psi_y);
        tma_prefetch_desc(&maps.psi_x); tma_prefetch_desc(&maps.u_c);   tma_prefetch_desc(&maps.u_z);
        tma_prefetch_desc(&maps.u_y);   tma_prefetch_desc(&maps.u_x);   tma_prefetch_desc(&maps.s_c);
        pol_n = l2_policy_evict_normal();
        pol_s = (prm.flags & 1) ? pol_n : l2_policy_evict_first();  // S is used exactly once
        pol_u = (prm.flags & 2) ? l2_policy_evict_first() : pol_n;
        pol_p = (prm.flags & 4) ? l2_policy_evict_last() : pol_n;
        nC = nR = nF = seq = 0;
        stage = ST_FETCH;
        g = j = t = 0;
        done = false;
    }
    __device__ __forceinline__ int pc() const { return 12 * ((g < ng) ? rhs0 + g : rhs0); }  // first component of group g's RHS
    __device__ __forceinline__ uint32_t gbase() const { return P::OFF_G + g * P::SZ_G; }
    __device__ __forceinline__ uint32_t gbar(int k) const { return 8 * (OB_GROUP + g * GB_COUNT + k); }

    // psi_g(tt) interior into group g's C buffer nC & 1
    __device__ __forceinline__ bool load_c(const TmaMaps &maps, uint32_t sbase, uint32_t bar_full, uint32_t bar_empty, int tt) {
        const uint32_t b = nC & 1, ob = gbar(GB_C + b);
        if (!mbar_try_wait(bar_empty + ob, ((nC >> 1) & 1) ^ 1)) return false;
        mbar_arrive_expect_tx(bar_full + ob, P::SZ_C);
        tma_load_5d_hint(sbase + gbase() + P::GO_C + b * P::SZ_C, &maps.psi_c, bar_full + ob, cx, y0, z0, tt, pc(), pol_p);
        return true;
    }
    // nine components of U or S into ring slot nR % kRing
    __device__ __forceinline__ bool load_ring(const CUtensorMap *map, uint32_t sbase, uint32_t bar_full, uint32_t bar_empty,
                                              int tt, int comp, uint64_t pol) {
        const uint32_t b = nR % kRing, ob = 8 * (OB_R + b);
        if (!mbar_try_wait(bar_empty + ob, ((nR / kRing) & 1) ^ 1)) return false;
        mbar_arrive_expect_tx(bar_full + ob, P::SZ_U);
        tma_load_5d_hint(sbase + P::OFF_R + b * P::SZ_U, map, bar_full + ob, cx, y0, z0, tt, comp, pol);
        nR++;
        return true;
    }
    // after a per-group object: next group, or on to `next` once all groups are served
    __device__ __forceinline__ void next_group(int next) {
        if (++g == P::G) {
            g = 0;
            stage = next;
        }
    }

    __device__ __forceinline__ bool advance(const TmaMaps &maps, const TmaParams &prm, unsigned char *smem, uint32_t sbase,
                                            uint32_t bar_full, uint32_t bar_empty) {
        constexpr int BZ = P::BZ, BY = P::BY, BX = P::BX;
        constexpr bool CLOVER = (P::SELF == SELF_CLOVER);
        if (done) return false;
        const int T = prm.n[0];
        const uint32_t pe = (nF & 1) ^ 1;
        const int tm1 = (t == 0) ? T - 1 : t - 1, tp1 = (t + 1 == T) ? 0 : t + 1;
        switch (stage) {
        case ST_FETCH: {
            const uint32_t slot = seq & 1, mpar = (seq >> 1) & 1;
            if (!mbar_try_wait(bar_empty + 8 * (OB_ITEM0 + slot), mpar ^ 1)) return false;
            const bool dynamic = !(prm.flags & 16);
            int item = dynamic ? (int)atomicAdd(prm.sched, 1u) : (int)(blockIdx.x + seq * gridDim.x);
            if (item >= prm.nitems) item = -1;
            reinterpret_cast<volatile int *>(smem + P::OFF_MAIL)[slot] = item;
            mbar_arrive(bar_full + 8 * (OB_ITEM0 + slot));
            seq++;
            if (item < 0) {
                if (dynamic && atomicAdd(prm.sched + 1, 1u) == gridDim.x - 1) {  // last CTA out re-arms the queue
                    prm.sched[0] = 0;
                    prm.sched[1] = 0;
                }
                done = true;
                return false;
            }
            const Item it = decode_item<P>(prm, item);
            const int Z = prm.n[1], Y = prm.n[2], X = prm.n[3];
            cx = 2 * it.x0, y0 = it.y0, z0 = it.z0;  // dim-0 coordinates count doubles
            rhs0 = it.rhs0, ng = it.ng;
            zlo = (z0 == 0) ? Z - 1 : z0 - 1, zhi = (z0 + BZ == Z) ? 0 : z0 + BZ;
            ylo = (y0 == 0) ? Y - 1 : y0 - 1, yhi = (y0 + BY == Y) ? 0 : y0 + BY;
            cxlo = 2 * ((it.x0 == 0) ? X - 1 : it.x0 - 1), cxhi = 2 * ((it.x0 + BX == X) ? 0 : it.x0 + BX);
            t = it.t0;
            j = 1;
            g = 0;
            stage = ST_PRO_C;
            return true;
        }
        case ST_PRO_C:  // psi_g(t0-1)
            if (!load_c(maps, sbase, bar_full, bar_empty, tm1)) return false;
            if (g == P::G - 1) nC++;
            next_group(ST_PRO_T);
            return true;
        case ST_PRO_T:  // U_T(t0-1)
            if (!load_ring(&maps.u_c, sbase, bar_full, bar_empty, tm1, 0, pol_u)) return false;
            stage = ST_PRO_C2;
            return true;
        case ST_PRO_C2:  // psi_g(t0)
            if (!load_c(maps, sbase, bar_full, bar_empty, t)) return false;
            if (g == P::G - 1) nC++;
            next_group(ST_UZ);
            return true;
        case ST_UZ:
            if (!mbar_try_wait(bar_empty + 8 * OB_UZ, pe)) return false;
            mbar_arrive_expect_tx(bar_full + 8 * OB_UZ, P::SZ_UZ);
            tma_load_5d_hint(sbase + P::OFF_UZ, &maps.u_c, bar_full + 8 * OB_UZ, cx, y0, z0, t, 9, pol_u);
            tma_load_5d_hint(sbase + P::OFF_UZF, &maps.u_z, bar_full + 8 * OB_UZ, cx, y0, zlo, t, 9, pol_u);
            stage = ST_PZ;
            return true;
        case ST_PZ:
            if (!mbar_try_wait(bar_empty + gbar(GB_PZ), pe)) return false;
            mbar_arrive_expect_tx(bar_full + gbar(GB_PZ), P::SZ_PZ);
            tma_load_5d_hint(sbase + gbase() + P::GO_ZLO, &maps.psi_z, bar_full + gbar(GB_PZ), cx, y0, zlo, t, pc(), pol_p);
            tma_load_5d_hint(sbase + gbase() + P::GO_ZHI, &maps.psi_z, bar_full + gbar(GB_PZ), cx, y0, zhi, t, pc(), pol_p);
            next_group(ST_UY);
            return true;
        case ST_UY:
            if (!mbar_try_wait(bar_empty + 8 * OB_UY, pe)) return false;
            mbar_arrive_expect_tx(bar_full + 8 * OB_UY, P::SZ_UY);
            tma_load_5d_hint(sbase + P::OFF_UY, &maps.u_c, bar_full + 8 * OB_UY, cx, y0, z0, t, 18, pol_u);
            tma_load_5d_hint(sbase + P::OFF_UYF, &maps.u_y, bar_full + 8 * OB_UY, cx, ylo, z0, t, 18, pol_u);
            stage = ST_PY;
            return true;
        case ST_PY:
            if (!mbar_try_wait(bar_empty + gbar(GB_PY), pe)) return false;
            mbar_arrive_expect_tx(bar_full + gbar(GB_PY), P::SZ_PY);
            tma_load_5d_hint(sbase + gbase() + P::GO_YLO, &maps.psi_y, bar_full + gbar(GB_PY), cx, ylo, z0, t, pc(), pol_p);
            tma_load_5d_hint(sbase + gbase() + P::GO_YHI, &maps.psi_y, bar_full + gbar(GB_PY), cx, yhi, z0, t, pc(), pol_p);
            next_group(CLOVER ? ST_S1 : ST_UX);
            return true;
        case ST_S1:
        case ST_S2:
        case ST_S3:
        case ST_S4:
            if (!load_ring(&maps.s_c, sbase, bar_full, bar_empty, t, 9 * (stage - ST_S1), pol_s)) return false;
            stage++;  // ... ST_S4 -> ST_UX
            return true;
        case ST_UX:
            if (!mbar_try_wait(bar_empty + 8 * OB_UX, pe)) return false;
            mbar_arrive_expect_tx(bar_full + 8 * OB_UX, P::SZ_UX);
            tma_load_5d_hint(sbase + P::OFF_UX, &maps.u_c, bar_full + 8 * OB_UX, cx, y0, z0, t, 27, pol_u);
            tma_load_5d_hint(sbase + P::OFF_UXF, &maps.u_x, bar_full + 8 * OB_UX, cxlo, y0, z0, t, 27, pol_u);
            stage = ST_PX;
            return true;
        case ST_PX:
            if (!mbar_try_wait(bar_empty + gbar(GB_PX), pe)) return false;
            mbar_arrive_expect_tx(bar_full + gbar(GB_PX), P::SZ_PX);
            tma_load_5d_hint(sbase + gbase() + P::GO_XLO, &maps.psi_x, bar_full + gbar(GB_PX), cxlo, y0, z0, t, pc(), pol_p);
            tma_load_5d_hint(sbase + gbase() + P::GO_XHI, &maps.psi_x, bar_full + gbar(GB_PX), cxhi, y0, z0, t, pc(), pol_p);
            next_group(ST_C);
            return true;
        case ST_C:  // psi_g(t+1)
            if (!load_c(maps, sbase, bar_full, bar_empty, tp1)) return false;
            if (g == P::G - 1) nC++;
            next_group(ST_T);
            return true;
        default:  // ST_T: U_T(t)
            if (!load_ring(&maps.u_c, sbase, bar_full, bar_empty, t, 0, pol_u)) return false;
            nF++;
            j++;
            t = tp1;
            stage = (j > prm.tchunk) ? ST_FETCH : ST_UZ;
            return true;
        }
    }
};

// ---------------------------------------------------------------- the kernel
template <class P>
__global__ void __launch_bounds__(P::NTHREADS, 1) k_tmr(const __grid_constant__ TmaMaps maps, const TmaParams prm) {
    extern __shared__ __align__(128) unsigned char smem[];
    const uint32_t sbase = smem_u32(smem);
    const uint32_t bar_full = sbase + P::OFF_BAR, bar_empty = bar_full + P::NBAR * 8;
    const int tid = threadIdx.x;
    constexpr int BZ = P::BZ, BY = P::BY, BX = P::BX, N = P::N, G = P::G;
    constexpr bool CLOVER = (P::SELF == SELF_CLOVER);

    if (tid == 0) {
        if (sbase & 127u) __trap();  // TMA destinations need 128-byte alignment
        for (int k = 0; k < P::NBAR; k++) {
            mbar_init(bar_full + 8 * k, 1);                               // the producer's arrive(.expect_tx)
            mbar_init(bar_empty + 8 * k, (k < OB_GROUP ? G : 1) * P::NW);  // shared objects: every group's warps
        }
        mbar_fence_init();
    }
    __syncthreads();

    const int T = prm.n[0], Z = prm.n[1], Y = prm.n[2], X = prm.n[3];

    if (tid >= G * N) {
        // ======================= producer: one thread issues every TMA =======================
        if (tid == G * N) {
            Producer<P> prod;
            prod.init(maps, prm);
            while (!prod.done) prod.advance(maps, prm, smem, sbase, bar_full, bar_empty);
        }
        return;
    }
    // ======================= consumers: group = right-hand side, thread = site =======================
    const int lane = tid & 31;
    const int grp = tid / N, stid = tid - grp * N;
    const int lx = stid % BX, ly = (stid / BX) % BY, lz = stid / (BX * BY);
    constexpr uint32_t E = P::E, NS = N * E;
    const uint32_t own = stid * E;
    const uint32_t gb = P::OFF_G + grp * P::SZ_G;  // this group's psi objects
    const uint32_t gbar = 8 * (OB_GROUP + grp * GB_COUNT);
    // operand addresses (bytes from the start of shared memory): interior (relative to the C buffer in use) or face
    const uint32_t fz = (ly * BX + lx) * E, fy = (lz * BX + lx) * E, fx = (lz * BY + ly) * E;
    const bool zf_in = lz < BZ - 1, zb_in = lz > 0, yf_in = ly < BY - 1, yb_in = ly > 0, xf_in = lx < BX - 1, xb_in = lx > 0;
    const uint32_t cbase = gb + P::GO_C + own;
    const uint32_t z_pf = zf_in ? cbase + P::FZ * E : gb + P::GO_ZHI + fz, z_pf_s = zf_in ? NS : P::FZ * E;
    const uint32_t z_pb = zb_in ? cbase - P::FZ * E : gb + P::GO_ZLO + fz, z_b_s = zb_in ? NS : P::FZ * E;
    const uint32_t z_ub = zb_in ? P::OFF_UZ + own - P::FZ * E : P::OFF_UZF + fz;
    const uint32_t y_pf = yf_in ? cbase + BX * E : gb + P::GO_YHI + fy, y_pf_s = yf_in ? NS : P::FY * E;
    const uint32_t y_pb = yb_in ? cbase - BX * E : gb + P::GO_YLO + fy, y_b_s = yb_in ? NS : P::FY * E;
    const uint32_t y_ub = yb_in ? P::OFF_UY + own - BX * E : P::OFF_UYF + fy;
    const uint32_t x_pf = xf_in ? cbase + E : gb + P::GO_XHI + fx, x_pf_s = xf_in ? NS : P::FX * E;
    const uint32_t x_pb = xb_in ? cbase - E : gb + P::GO_XLO + fx, x_b_s = xb_in ? NS : P::FX * E;
    const uint32_t x_ub = xb_in ? P::OFF_UX + own - E : P::OFF_UXF + fx;

    auto release = [&](uint32_t bar8) {  // bar8 = 8 * barrier index
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + bar8);
    };
    auto wait_full = [&](uint32_t bar8, uint32_t parity) { mbar_wait(bar_full + bar8, parity); };

    const long long V = prm.Vs;  // component stride
    const long long strideT = (long long)Z * Y * X;
    uint32_t nC = 0, nR = 0, nF = 0;  // fills consumed so far: C buffers, ring slots, per-step objects
    cd acc[12];

    // one 6x6 block of S (two consecutive ring objects): acc[6b..6b+5] += B_b * (-2 psi)
    auto s_phase = [&](uint32_t cb, int b, bool active) {
        const uint32_t s0 = nR % kRing, s1 = (nR + 1) % kRing;
        wait_full(8 * (OB_R + s0), (nR / kRing) & 1);
        wait_full(8 * (OB_R + s1), ((nR + 1) / kRing) & 1);
        if (active) {
            cd q[6];
#pragma unroll
            for (int c = 0; c < 6; c++) {
                const cd v = lds(smem, cbase + cb + (6 * b + c) * NS);
                q[c] = make_double2(-2.0 * v.x, -2.0 * v.y);
            }
            herm6_half_add<0>(acc + 6 * b, smem, P::OFF_R + s0 * P::SZ_U + own, NS, q);
            herm6_half_add<1>(acc + 6 * b, smem, P::OFF_R + s1 * P::SZ_U + own, NS, q);
        }
        release(8 * (OB_R + s0));
        release(8 * (OB_R + s1));
        nR += 2;
    };

    const volatile int *mail = reinterpret_cast<const volatile int *>(smem + P::OFF_MAIL);
    for (uint32_t seq = 0;; seq++) {
        const uint32_t mslot = seq & 1, mpar = (seq >> 1) & 1;
        wait_full(8 * (OB_ITEM0 + mslot), mpar);
        const int item = mail[mslot];
        release(8 * (OB_ITEM0 + mslot));
        if (item < 0) break;
        const Item it = decode_item<P>(prm, item);
        const bool active = grp < it.ng;  // else: go through the barriers only
        const long long site0 = ((long long)(it.z0 + lz) * Y + (it.y0 + ly)) * X + (it.x0 + lx);
        cd *__restrict__ out = prm.out + (long long)(it.rhs0 + (active ? grp : 0)) * 12 * V;
        int t = it.t0;
        {   // prologue: acc = backward-T hop of slice t0, (1 + gamma_T) U_T(t0-1)^H psi(t0-1)
            const uint32_t cb = (nC & 1) ? P::SZ_C : 0, slot = nR % kRing;
            wait_full(gbar + 8 * (GB_C + (nC & 1)), (nC >> 1) & 1);
            wait_full(8 * (OB_R + slot), (nR / kRing) & 1);
            cd p[12], u[9], h[6], g[6];
#pragma unroll
            for (int k = 0; k < 9; k++) u[k] = lds(smem, P::OFF_R + slot * P::SZ_U + own + k * NS);
#pragma unroll
            for (int c = 0; c < 12; c++) p[c] = lds(smem, cbase + cb + c * NS);
            release(gbar + 8 * (GB_C + (nC & 1)));
            release(8 * (OB_R + slot));
            nC++;
            nR++;
            project<0, +1>(h, p);
            su3_mul<true>(g, u, h);
#pragma unroll
            for (int c = 0; c < 12; c++) acc[c] = make_double2(0.0, 0.0);
            reconstruct_add<0, +1>(acc, g);
        }
        for (int j = 1; j <= prm.tchunk; j++) {
            const bool last = (j == prm.tchunk);
            const uint32_t cb = (nC & 1) ? P::SZ_C : 0;  // C buffer holding psi(t)
            if (j == 1) wait_full(gbar + 8 * (GB_C + (nC & 1)), (nC >> 1) & 1);
            const uint32_t pf = nF & 1;
            wait_full(8 * OB_UZ, pf);
            wait_full(gbar + 8 * GB_PZ, pf);
            if (active)
                hop_pair_smem<1>(acc, smem, P::OFF_UZ + own, NS, z_pf + (zf_in ? cb : 0), z_pf_s, z_ub, z_b_s,
                                 z_pb + (zb_in ? cb : 0), z_b_s);
            release(8 * OB_UZ);
            release(gbar + 8 * GB_PZ);
            wait_full(8 * OB_UY, pf);
            wait_full(gbar + 8 * GB_PY, pf);
            if (active)
                hop_pair_smem<2>(acc, smem, P::OFF_UY + own, NS, y_pf + (yf_in ? cb : 0), y_pf_s, y_ub, y_b_s,
                                 y_pb + (yb_in ? cb : 0), y_b_s);
            release(8 * OB_UY);
            release(gbar + 8 * GB_PY);
            if (CLOVER) {
                s_phase(cb, 0, active);
                s_phase(cb, 1, active);
            }
            wait_full(8 * OB_UX, pf);
            wait_full(gbar + 8 * GB_PX, pf);
            if (active)
                hop_pair_smem<3>(acc, smem, P::OFF_UX + own, NS, x_pf + (xf_in ? cb : 0), x_pf_s, x_ub, x_b_s,
                                 x_pb + (xb_in ? cb : 0), x_b_s);
            release(8 * OB_UX);
            release(gbar + 8 * GB_PX);
            nF++;
            {   // T phase: forward hop completes out(t); the backward hop of slice t+1 starts the next accumulator
                const uint32_t cn = cb ^ P::SZ_C, slot = nR % kRing;  // psi(t+1) is in the other C buffer
                wait_full(gbar + 8 * (GB_C + ((nC + 1) & 1)), ((nC + 1) >> 1) & 1);
                wait_full(8 * (OB_R + slot), (nR / kRing) & 1);
                if (active) {
                    cd u[9], p[12];
#pragma unroll
                    for (int k = 0; k < 9; k++) u[k] = lds(smem, P::OFF_R + slot * P::SZ_U + own + k * NS);
#pragma unroll
                    for (int c = 0; c < 12; c++) p[c] = lds(smem, cbase + cn + c * NS);
                    hop_term<0, -1>(acc, p, u);
                    if (P::SELF == SELF_MASS || !last) {
#pragma unroll
                        for (int c = 0; c < 12; c++) p[c] = lds(smem, cbase + cb + c * NS);  // psi(t)
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
#pragma unroll
                        for (int c = 0; c < 12; c++) acc[c] = make_double2(0.0, 0.0);
                        reconstruct_add<0, +1>(acc, g);
                    }
                }
                release(8 * (OB_R + slot));
                nR++;
                release(gbar + 8 * (GB_C + (nC & 1)));  // psi(t) is done; psi(t+1) stays for the next step
                nC++;
                if (last) {                              // ... unless this was the item's last slice
                    release(gbar + 8 * (GB_C + (nC & 1)));
                    nC++;
                }
            }
            t = (t + 1 == T) ? 0 : t + 1;
        }
    }
}

// ---------------------------------------------------------------- host side
static int sm_count() {  // of the current device
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1)
        n = 148;
    return n;
}

// Work decomposition: an item = (T chunk, block of G right-hand sides, tile).  Short chunks and a compact panel
// of tiles in flight, as in wd_tmb.cu.
template <class P> static void plan_items(const KParams &p, TmaParams &prm) {
    const int nsm = sm_count();
    prm.ntx = p.n[3] / P::BX;
    prm.nty = p.n[2] / P::BY;
    prm.ntz = p.n[1] / P::BZ;
    const int ntiles = prm.ntx * prm.nty * prm.ntz, T = p.n[0];
    int best_tc = T;
    if (p.opt_tchunk > 0 && T % p.opt_tchunk == 0) {
        best_tc = p.opt_tchunk;
    } else {
        best_tc = 1;
        for (int tc = 1; tc <= T && tc <= 16; tc++)
            if (T % tc == 0) best_tc = tc;
        if (best_tc < 4 && T > 16) best_tc = T;
    }
    prm.tchunk = best_tc;
    prm.ntc = T / best_tc;
    prm.nrhs = p.nrhs;
    prm.nblk = (p.nrhs + P::G - 1) / P::G;
    prm.nitems = ntiles * prm.ntc * prm.nblk;
    int bpy = 1, bpz = 1;
    double bscore = 1e300;
    for (int py = 1; py <= prm.nty; py++) {
        if (prm.nty % py) continue;
        for (int pz = 1; pz <= prm.ntz; pz++) {
            if (prm.ntz % pz) continue;
            if (p.opt_zgroup > 0 && pz != p.opt_zgroup && prm.ntz % p.opt_zgroup == 0) continue;
            const int tiles = prm.ntx * py * pz;
            double score = 1.0 / (py * P::BY) + 1.0 / (pz * P::BZ);
            if (tiles > nsm) score += 10.0 * tiles / nsm;  // over one wave: only if nothing smaller exists
            if (score < bscore) bscore = score, bpy = py, bpz = pz;
        }
    }
    prm.py = bpy;
    prm.pz = bpz;
}

template <int BZ, int BY, int BX, int SELF, int G> static cudaError_t launch_self(const KParams &p, cudaStream_t st) {
    using P = Plan<BZ, BY, BX, SELF, G>;
    static bool attr_done[64] = {};  // per device: the attribute belongs to the device's copy of the kernel
    int dev_id = 0;
    cudaGetDevice(&dev_id);
    if (dev_id < 0 || dev_id >= 64 || !attr_done[dev_id]) {
        cudaError_t e0 = cudaFuncSetAttribute(k_tmr<P>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)P::SMEM);
        if (e0 != cudaSuccess) return e0;
        if (dev_id >= 0 && dev_id < 64) attr_done[dev_id] = true;
    }
    TmaMaps maps;
    cudaError_t e;
#define WD_ENC(m, base, nc, bx, by, bz, bc)                                      \
    if ((e = encode_field_map(&maps.m, base, p.n, p.Vs, nc, bx, by, bz, bc)) != cudaSuccess) return e;
    WD_ENC(psi_c, p.psi, 12 * p.nrhs, BX, BY, BZ, 12)
    WD_ENC(psi_z, p.psi, 12 * p.nrhs, BX, BY, 1, 12)
    WD_ENC(psi_y, p.psi, 12 * p.nrhs, BX, 1, BZ, 12)
    WD_ENC(psi_x, p.psi, 12 * p.nrhs, 1, BY, BZ, 12)
    WD_ENC(u_c, p.U, 36, BX, BY, BZ, 9)
    WD_ENC(u_z, p.U, 36, BX, BY, 1, 9)
    WD_ENC(u_y, p.U, 36, BX, 1, BZ, 9)
    WD_ENC(u_x, p.U, 36, 1, BY, BZ, 9)
    WD_ENC(s_c, (SELF == SELF_CLOVER) ? p.S : p.U, 36, BX, BY, BZ, 9)
#undef WD_ENC
    TmaParams prm;
    prm.out = p.out;
    prm.V = p.V;
    prm.Vs = p.Vs;
    for (int a = 0; a < 4; a++) prm.n[a] = p.n[a];
    prm.mass = p.mass;
    plan_items<P>(p, prm);
    const int grid = (prm.nitems < sm_count()) ? prm.nitems : sm_count();
    prm.sched = p.sched;
    prm.flags = getenv("WD_TMA_FLAGS") ? atoi(getenv("WD_TMA_FLAGS")) : 0;
    k_tmr<P><<<grid, P::NTHREADS, P::SMEM, st>>>(maps, prm);
    return cudaGetLastError();
}

template <int BZ, int BY, int BX, int G> static cudaError_t launch(const KParams &p, int self, cudaStream_t st) {
    if (self == SELF_CLOVER) return launch_self<BZ, BY, BX, SELF_CLOVER, G>(p, st);
    if (self == SELF_MASS) return launch_self<BZ, BY, BX, SELF_MASS, G>(p, st);
    return launch_self<BZ, BY, BX, SELF_NONE, G>(p, st);
}
}  // namespace tmr

cudaError_t launch_tmr_2x4x8_g3(const KParams &p, int self, cudaStream_t st) { return tmr::launch<2, 4, 8, 3>(p, self, st); }
cudaError_t launch_tmr_2x4x8_g2(const KParams &p, int self, cudaStream_t st) { return tmr::launch<2, 4, 8, 2>(p, self, st); }
}  // namespace wd
