// wd_tma_common.cuh — the ONE skeleton shared by the TMA-staged T-marching kernels (wd_tma.cu, wd_tmb.cu): tensor maps and their per-handle cache, launch parameters, the work-item order, the work
// decomposition (T chunk, rasterisation panel) and the launch wrapper.  A kernel file only adds its
// shared-memory plan, its producer and its consumer code.
//
// Work item = (T chunk, unit of G right-hand sides, tile).  The CTA that takes an item marches the tile
// along T for `tchunk` slices.  Items are handed out by an atomic queue (fast SMs take more; the measured
// SM-to-SM spread of the streaming rate is ~20 %, profiles/r1b), the last CTA out re-arms the queue.
#pragma once
#include <mutex>

#include "wd_internal.h"
#include "wd_math.cuh"
#include "wd_tma.cuh"

namespace wd {

struct TmaMaps {
    CUtensorMap psi_c, psi_z, psi_y, psi_x;  // boxes: interior, z-face, y-face, x-face (12 components)
    CUtensorMap u_c, u_z, u_y, u_x;          // same shapes, one link (9 components; 6 with two-row storage)
    CUtensorMap s_c;                         // interior box of S: 18 components (a 6x6 block) or 9 (half of one)
};

struct TmaParams {
    void *out;              // double2 (or float2, FP32 variant) [nrhs][12][Vs]
    const double2 *psi, *U, *S;  // the fields themselves (kernels that read operands with LDG)
    long long V, Vs;       // sites, component stride
    int n[4];
    int ntx, nty, ntz;     // tiles per direction
    int py, pz;            // rasterisation panel (in tiles); py | nty, pz | ntz
    int tchunk, ntc;       // T steps per work item, items per tile
    int nrhs;              // right-hand sides in this launch
    int nunits, rb;        // units of G right-hand sides; units per block of the item order
    int chunk0;            // first T chunk of this launch (0 unless a T range was asked for)
    int nitems;            // ntx*nty*ntz*(chunks of this launch)*nunits
    int open_mask;         // bit mu set: direction mu does NOT wrap (domain-decomposed sub-lattice, wd_dd.cu):
                           // hops across that boundary are left out (the exterior kernel adds them)
    double mass;
    unsigned int *sched;   // [0] next item, [1] CTAs finished (both 0 between launches)
#ifdef WD_EXPERIMENTS
    int flags;             // WD_TMA_FLAGS: 1 S evict_normal instead of evict_first, 2 U evict_first, 4 psi evict_last,
                           // 8 L2-prefetch psi(t+1), 16 static round-robin items
    unsigned long long *trace;  // WD_TMA_TRACE: [cta][kTraceLen] globaltimer per step, or null
#endif
};
constexpr int kTraceLen = 1024;

#ifdef WD_EXPERIMENTS
#define WD_FLAG(prm, bit) ((prm).flags & (bit))
#else
#define WD_FLAG(prm, bit) 0
#endif

struct Item {
    int x0, y0, z0, t0;
    int rhs0, ng;  // first right-hand side of the unit, number of right-hand sides in it (<= G)
};

// Item order (slowest to fastest): T chunk, block of up to `rb` units, tile (panel order), unit within the
// block.  The CTAs in flight therefore work on the same few tiles for rb units at once: the links and S of a
// tile are fetched from HBM by the first of them and are L2 hits for the others (a8: +384 B per extra RHS
// instead of +1536 B).
template <class P> __device__ __forceinline__ Item decode_item(const TmaParams &prm, int item) {
    const int ntiles = prm.ntx * prm.nty * prm.ntz;
    const int per_chunk = ntiles * prm.nunits;
    const int chunk_rel = item / per_chunk;
    const int chunk = chunk_rel + prm.chunk0;
    int rem = item - chunk_rel * per_chunk;
    const int blk = rem / (ntiles * prm.rb);
    rem -= blk * ntiles * prm.rb;
    const int rb_here = min(prm.rb, prm.nunits - blk * prm.rb);
    const int tile = rem / rb_here;
    const int unit = blk * prm.rb + (rem - tile * rb_here);
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
    it.rhs0 = unit * P::G;
    it.ng = min(P::G, prm.nrhs - it.rhs0);
    return it;
}

// The producer's queue access: next item or -1; the last CTA to run dry re-arms the queue for the next launch.
__device__ __forceinline__ int fetch_item(const TmaParams &prm, uint32_t seq) {
    const bool dynamic = !WD_FLAG(prm, 16);
    int item = dynamic ? (int)atomicAdd(prm.sched, 1u) : (int)(blockIdx.x + seq * gridDim.x);
    if (item >= prm.nitems) item = -1;
    if (item < 0 && dynamic && atomicAdd(prm.sched + 1, 1u) == gridDim.x - 1) {
        prm.sched[0] = 0;
        prm.sched[1] = 0;
    }
    return item;
}

// ---------------------------------------------------------------- host side
// Tensor maps depend only on (field pointers, nrhs, tile): cached per handle so that wd_apply does no
// cuTensorMapEncodeTiled calls in steady state (0.26 ms applies at 32^4, GMRES loops).
struct MapCache {
    struct Entry {
        int tag;  // kernel family and tile
        const void *psi, *U, *S;
        int nrhs;
        TmaMaps maps;
    };
    static constexpr int kEntries = 80;  // a GMRES(m) cycle applies the operator to m + 2 <= 66 different vectors, in cyclic
                                         // order (round-robin eviction of fewer entries would miss on every one); the rest
                                         // is for the caller's own buffers
    Entry e[kEntries];
    int used = 0, next = 0;
    const TmaMaps *find(int tag, const void *psi, const void *U, const void *S, int nrhs) const {
        for (int k = 0; k < used; k++)
            if (e[k].tag == tag && e[k].psi == psi && e[k].U == U && e[k].S == S && e[k].nrhs == nrhs) return &e[k].maps;
        return nullptr;
    }
    TmaMaps *insert(int tag, const void *psi, const void *U, const void *S, int nrhs) {
        const int k = (used < kEntries) ? used++ : (next++ % kEntries);
        e[k].tag = tag, e[k].psi = psi, e[k].U = U, e[k].S = S, e[k].nrhs = nrhs;
        return &e[k].maps;
    }
    void clear() { used = next = 0; }
};

enum ChunkPolicy {
    CHUNK_COST_MODEL,  // minimise items*(tchunk + 1/2)/SMs + (tchunk + 1)/2   (first generation)
    CHUNK_SHORT        // largest divisor of T up to 16: CTAs of a panel stay within a few steps of each other
};

// Work decomposition.  tchunk trades the tail (the last items finish unevenly) against the per-item
// prologue/epilogue (one extra psi slice in, one extra psi + U_T slice at the end).  The panel (py x pz
// tiles, all of X) is the set of tiles in flight together: as cubic as possible, at most one wave, so that
// most face re-reads are L2 hits on data a neighbouring CTA is streaming at the same time.
template <class P> static void plan_items(const KParams &p, TmaParams &prm, ChunkPolicy policy, int rb_units) {
    const int nsm = p.nsm * P::CTAS_PER_SM;  // persistent CTAs in flight
    prm.ntx = p.n[3] / P::BX;
    prm.nty = p.n[2] / P::BY;
    prm.ntz = p.n[1] / P::BZ;
    prm.nrhs = p.nrhs;
    prm.nunits = (p.nrhs + P::G - 1) / P::G;
    const int ntiles = prm.ntx * prm.nty * prm.ntz, T = p.n[0];
    int best_tc = T;
    if (p.opt_tchunk > 0 && T % p.opt_tchunk == 0) {
        best_tc = p.opt_tchunk;
    } else if (policy == CHUNK_COST_MODEL) {
        double best = 1e300;
        for (int tc = 1; tc <= T; tc++) {
            if (T % tc) continue;
            const long long items = (long long)ntiles * (T / tc) * prm.nunits;
            const double cost = (double)items * (tc + 0.5) / nsm + 0.5 * (tc + 1);
            if (cost < best * 0.999) best = cost, best_tc = tc;
        }
    } else {
        best_tc = 1;
        for (int tc = 1; tc <= T && tc <= 16; tc++)
            if (T % tc == 0) best_tc = tc;
        if (best_tc < 4 && T > 16) best_tc = T;  // T without a small divisor: one chunk
    }
    prm.tchunk = best_tc;
    prm.ntc = T / best_tc;
    prm.rb = (prm.nunits < rb_units) ? prm.nunits : rb_units;
#ifdef WD_EXPERIMENTS
    if (const char *e = getenv("WD_TMA_RB")) {
        const int v = atoi(e);
        if (v >= 1) prm.rb = (v < prm.nunits) ? v : prm.nunits;
    }
#endif
    prm.chunk0 = (p.tc_count > 0) ? p.tc_begin : 0;
    prm.nitems = ntiles * ((p.tc_count > 0) ? p.tc_count : prm.ntc) * prm.nunits;
    const int wave = (nsm / prm.rb > 0) ? nsm / prm.rb : 1;  // tiles in flight together
    int bpy = 1, bpz = 1;
    double bscore = 1e300;
    for (int py = 1; py <= prm.nty; py++) {
        if (prm.nty % py) continue;
        for (int pz = 1; pz <= prm.ntz; pz++) {
            if (prm.ntz % pz) continue;
            if (p.opt_zgroup > 0 && pz != p.opt_zgroup && prm.ntz % p.opt_zgroup == 0) continue;
            const int tiles = prm.ntx * py * pz;
            double score = 1.0 / (py * P::BY) + 1.0 / (pz * P::BZ);
            if (tiles > wave) score += 10.0 * tiles / wave;  // over one wave: only if nothing smaller exists
            if (score < bscore) bscore = score, bpy = py, bpz = pz;
        }
    }
    prm.py = bpy;
    prm.pz = bpz;
}

// Tensor maps of one launch: from the handle's cache, encoded on a miss.  ucomp = components per link box
// (9, or 6 with two-row storage), scomp = components per S box (18 or 9).
template <class P> static cudaError_t get_maps(const KParams &p, int ucomp, int scomp, const TmaMaps **out, TmaMaps *scratch) {
    constexpr int BZ = P::BZ, BY = P::BY, BX = P::BX;
    static_assert(BZ < 16 && BY < 32 && BX < 64 && P::G < 16, "tag fields");
    const int tag = ((((((ucomp * 32 + scomp) * 16 + BZ) * 32 + BY) * 64 + BX) * 16 + P::G) * 2 + (p.esize == 8)) * 2 + P::BLK;  // everything a box depends on
    const void *Sbase = (P::SELF == SELF_CLOVER) ? (const void *)p.S : (const void *)p.U;
    if (p.maps) {
        if (const TmaMaps *m = p.maps->find(tag, p.psi, p.U, Sbase, p.nrhs)) {
            *out = m;
            return cudaSuccess;
        }
    }
    TmaMaps *maps = p.maps ? p.maps->insert(tag, p.psi, p.U, Sbase, p.nrhs) : scratch;
    cudaError_t e;
    const int nucomp = 4 * ucomp, nscomp = (P::SELF == SELF_CLOVER) ? 36 : nucomp;
    const int sc = (scomp <= nscomp) ? scomp : nscomp;
#define WD_ENC(m, base, nc, bx, by, bz, bc) WD_ENCR(m, base, nc, bx, by, bz, bc, 1)
#define WD_ENCR(m, base, nc, bx, by, bz, bc, rb)                                             \
    if ((e = encode_field_map(&maps->m, base, p.n, p.Vs, nc, bx, by, bz, bc, p.esize, rb)) != cudaSuccess) { \
        if (p.maps) p.maps->clear();                                                         \
        return e;                                                                            \
    }
    // spinor boxes: the G right-hand sides of a unit — 12 G consecutive components of the plain layout, or 12 components of
    // G-interleaved sites in the blocked layout (whose units are padded to G right-hand sides)
    const int pcomp = P::BLK ? 12 * ((p.nrhs + P::G - 1) / P::G) : 12 * p.nrhs, pbox = P::BLK ? 12 : 12 * P::G;
    WD_ENCR(psi_c, p.psi, pcomp, BX, BY, BZ, pbox, P::RBK)
    WD_ENCR(psi_z, p.psi, pcomp, BX, BY, 1, pbox, P::RBK)
    WD_ENCR(psi_y, p.psi, pcomp, BX, 1, BZ, pbox, P::RBK)
    WD_ENCR(psi_x, p.psi, pcomp, P::XW, BY, BZ, pbox, P::RBK)
    WD_ENC(u_c, p.U, nucomp, BX, BY, BZ, ucomp)
    WD_ENC(u_z, p.U, nucomp, BX, BY, 1, ucomp)
    WD_ENC(u_y, p.U, nucomp, BX, 1, BZ, ucomp)
    WD_ENC(u_x, p.U, nucomp, P::XW, BY, BZ, ucomp)
    WD_ENC(s_c, Sbase, nscomp, BX, BY, BZ, sc)
#undef WD_ENC
#undef WD_ENCR
    *out = maps;
    return cudaSuccess;
}

// cudaFuncAttributeMaxDynamicSharedMemorySize belongs to the device's copy of the kernel: once per (kernel, device).
// (All kernels share one signature, hence one instantiation of this template: the table is keyed by the pointer.)
template <class K> static cudaError_t ensure_smem_attr(K kernel, int smem, int device) {
    struct Done {
        const void *fn;
        int device;
    };
    static std::mutex mu;
    static Done done[256];
    static int ndone = 0;
    std::lock_guard<std::mutex> lock(mu);
    for (int k = 0; k < ndone; k++)
        if (done[k].fn == (const void *)kernel && done[k].device == device) return cudaSuccess;
    const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e == cudaSuccess && ndone < 256) done[ndone++] = Done{(const void *)kernel, device};
    return e;
}

// The launch wrapper: attribute, maps, work decomposition, one persistent CTA per SM.
template <class P, class K>
static cudaError_t launch_tma_kernel(K kernel, const KParams &p, cudaStream_t st, int ucomp, int scomp,
                                     ChunkPolicy policy, int rb_units) {
    cudaError_t e = ensure_smem_attr(kernel, (int)P::SMEM, p.device);
    if (e != cudaSuccess) return e;
    TmaMaps scratch;
    const TmaMaps *maps = nullptr;
    if ((e = get_maps<P>(p, ucomp, scomp, &maps, &scratch)) != cudaSuccess) return e;
    TmaParams prm;
    prm.out = p.out;
    prm.psi = p.psi;
    prm.U = p.U;
    prm.S = p.S;
    prm.V = p.V;
    prm.Vs = p.Vs;
    for (int a = 0; a < 4; a++) prm.n[a] = p.n[a];
    prm.mass = p.mass;
    prm.open_mask = p.open_mask;
    plan_items<P>(p, prm, policy, rb_units);
    const int ctas = p.nsm * P::CTAS_PER_SM;
    const int grid = (prm.nitems < ctas) ? prm.nitems : ctas;
    if (grid < 1) return cudaSuccess;
    prm.sched = p.sched;
#ifdef WD_EXPERIMENTS
    prm.flags = getenv("WD_TMA_FLAGS") ? atoi(getenv("WD_TMA_FLAGS")) : 0;
    prm.trace = nullptr;
    const char *trace_path = getenv("WD_TMA_TRACE");
    if (trace_path) {
        if ((e = cudaMalloc((void **)&prm.trace, (size_t)grid * kTraceLen * 8)) != cudaSuccess) return e;
        cudaMemsetAsync(prm.trace, 0, (size_t)grid * kTraceLen * 8, st);
    }
#endif
    kernel<<<grid, P::NTHREADS, P::SMEM, st>>>(*maps, prm);
    e = cudaGetLastError();
#ifdef WD_EXPERIMENTS
    if (trace_path && e == cudaSuccess) {  // diagnostics only: synchronous dump of the last launch's step times
        unsigned long long *host = (unsigned long long *)malloc((size_t)grid * kTraceLen * 8);
        cudaStreamSynchronize(st);
        cudaMemcpy(host, prm.trace, (size_t)grid * kTraceLen * 8, cudaMemcpyDeviceToHost);
        if (FILE *f = fopen(trace_path, "wb")) {
            const int hdr[4] = {grid, kTraceLen, prm.tchunk, prm.nitems};
            fwrite(hdr, sizeof(int), 4, f);
            fwrite(host, 8, (size_t)grid * kTraceLen, f);
            fclose(f);
        }
        free(host);
    }
    if (prm.trace) cudaFree(prm.trace);
#endif
    return e;
}

}  // namespace wd
