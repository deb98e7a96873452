"""GPU parity of the domain-decomposed operator (csrc/wd_dd.cu + open-boundary mode of the fused kernels): 2, 4 and 8
sub-lattices on ONE device, the half-spinor faces exchanged through device buffers, compared with the oracle's
operator on the undivided global lattice (rel. L2 <= 1e-13).  Only one GPU is reachable per run, so this is how the
decomposition is proven; the rank arithmetic and the exchange order are covered on the CPU (test_decomposition.py)."""
import numpy as np
import pytest

import oracle
import paper_2407_00041_b200 as wd
import wdinputs
from latticeutil import rel_l2
from paper_2407_00041_b200.dd import EmulatedDecomposition
from test_gpu_parity import TOL, torch  # noqa: F401  (fixture)

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("gdims,grid", [
    ((8, 8, 8, 16), (2, 1, 1, 1)),    # T split in two (both neighbours are the same rank)
    ((16, 4, 8, 16), (4, 1, 1, 1)),   # T split in four
    ((8, 8, 8, 16), (2, 2, 1, 1)),    # T and Z (the 8-GPU plan of DESIGN.md at a small size)
    ((4, 8, 8, 32), (1, 2, 2, 2)),    # Z, Y and X
    ((8, 4, 8, 32), (2, 2, 2, 1)),    # eight sub-lattices
    ((6, 6, 4, 6), (2, 3, 1, 1)),     # odd local extents: only the linear LDG kernel fits
    ((2, 4, 4, 16), (2, 1, 1, 1)),    # local T extent 1: high and low face are the same sites
])
def test_decomposed_operator_matches_oracle_on_the_global_lattice(torch, gdims, grid):
    m0, csw, nrhs = -0.4, 1.0, 2
    U = wdinputs.gauge_haar(gdims, 801)
    psi = wdinputs.spinor(gdims, 802, nrhs=nrhs)
    C = oracle.build_clover(gdims, m0, csw, U)
    ref_c = oracle.apply(gdims, m0, U, C, psi)
    ref_w = oracle.apply(gdims, m0, U, None, psi)
    em = EmulatedDecomposition(torch, gdims, grid, m0, csw, U, C)  # S cut out of the oracle's global field
    try:
        kname = wd.wd_kernel_name(wd.wd_kernel_in_use(em.ops[0].h))
        assert rel_l2(em.apply(psi, nrhs), ref_c) <= TOL, kname
    finally:
        em.close()
    em = EmulatedDecomposition(torch, gdims, grid, m0, 0.0, U)  # pure Wilson
    try:
        assert rel_l2(em.apply(psi, nrhs), ref_w) <= TOL
    finally:
        em.close()


@pytest.mark.parametrize("kernel", ["tmw_2x4x16", "tma_2x4x16", "tmb_4x4x8", "tmq_2x4x8", "tile_1x4x4x16", "linear256"])
def test_every_kernel_family_supports_open_boundaries(torch, kernel):
    gdims, grid, m0, csw = (8, 8, 16, 32), (2, 2, 1, 2), -0.4, 1.0
    U = wdinputs.gauge_exp(gdims, 811, 0.5)
    psi = wdinputs.spinor(gdims, 812)
    C = wdinputs.selfcoupling_random(gdims, 813)
    ref = oracle.apply(gdims, m0, U, C, psi)
    em = EmulatedDecomposition(torch, gdims, grid, m0, csw, U, C)
    try:
        for op in em.ops:
            wd.wd_set_option(op.h, wd.WD_OPT_KERNEL, wd.kernel_id(kernel))
        assert rel_l2(em.apply(psi), ref) <= TOL
    finally:
        em.close()


def test_quad_kernel_on_sub_lattices_with_several_right_hand_sides(torch):
    """tmq_2x4x8 (one thread per site and right-hand side) with open boundaries in T, Z and X, five right-hand sides (a full
    unit of four and a partial one) through pack / exchange / interior / exterior."""
    gdims, grid, m0, csw, nrhs = (8, 8, 16, 32), (2, 2, 1, 2), -0.4, 1.0, 5
    U = wdinputs.gauge_exp(gdims, 831, 0.5)
    psi = wdinputs.spinor(gdims, 832, nrhs=nrhs)
    C = wdinputs.selfcoupling_random(gdims, 833)
    ref = oracle.apply(gdims, m0, U, C, psi)
    em = EmulatedDecomposition(torch, gdims, grid, m0, csw, U, C)
    try:
        for op in em.ops:
            wd.wd_set_option(op.h, wd.WD_OPT_KERNEL, wd.kernel_id("tmq_2x4x8"))
        out = em.apply(psi, nrhs)
        for r in range(nrhs):
            assert rel_l2(out[r], ref[r]) <= TOL, r
    finally:
        em.close()


def test_local_clover_from_extended_links_and_state_rules(torch):
    """S of a sub-lattice built on the device from the links of the local lattice extended by one site, against the
    oracle's S of the global lattice; wd_build_clover is refused on a decomposed handle."""
    gdims, grid, m0, csw = (8, 8, 4, 16), (2, 2, 1, 1), -0.4, 1.0
    U = wdinputs.gauge_exp(gdims, 821, 0.4)
    psi = wdinputs.spinor(gdims, 822)
    C = oracle.build_clover(gdims, m0, csw, U)
    em = EmulatedDecomposition(torch, gdims, grid, m0, csw, U)  # C_global = None: local_clover path
    try:
        for r, op in enumerate(em.ops):
            Cl = np.empty((int(np.prod(em.decomp.local_dims)), 42, 2))
            wd.wd_get_clover(op.h, Cl)
            assert rel_l2(Cl, em.decomp.extract(C, r)) <= TOL
            with pytest.raises(wd.WDError) as e:
                wd.wd_build_clover(op.h)
            assert e.value.code == wd.WD_ESTATE
            assert wd.wd_dd_open_mask(op.h) == 0b0011 and wd.wd_dd_face_sites(op.h, 2) == 0
            with pytest.raises(wd.WDError):
                wd.wd_dd_pack(op.h, op.spinor(), 1, 2, op.spinor(), op.spinor())  # Y is not decomposed
        assert rel_l2(em.apply(psi), oracle.apply(gdims, m0, U, C, psi)) <= TOL
    finally:
        em.close()
    with pytest.raises(wd.WDError):
        wd.wd_create_local((8, 8, 8, 8), (3, 1, 1, 1), (0, 0, 0, 0), 0.0, 0.0)


def test_decomposed_bench_size_slab(torch, capsys):
    """The 8-GPU plan of the bench (64^4 cut 4 x 2 in T and Z: local 16 x 32 x 64 x 64) on one sub-lattice pair:
    a 32 x 32 x 64 x 64 global lattice cut (2, 1, 1, 1), default kernels, compared with the oracle on every site."""
    gdims, grid, m0, csw = (32, 32, 64, 64), (2, 1, 1, 1), -0.4, 1.0
    U = wdinputs.gauge_haar(gdims, 831)
    psi = wdinputs.spinor(gdims, 832)
    C = oracle.build_clover(gdims, m0, csw, U)
    ref = oracle.apply(gdims, m0, U, C, psi)
    em = EmulatedDecomposition(torch, gdims, grid, m0, csw, U, C)
    try:
        out = em.apply(psi)
        kname = wd.wd_kernel_name(wd.wd_kernel_in_use(em.ops[0].h))
    finally:
        em.close()
    err = rel_l2(out, ref)
    with capsys.disabled():
        print(f"\n[decomposed parity] global {'x'.join(map(str, gdims))} grid {grid} kernel {kname}: rel_l2 {err:.3e}", flush=True)
    assert err <= TOL


class _InProcessDist:
    """Stand-in for torch.distributed point-to-point between `world` ranks that are THREADS of this process sharing one
    GPU: a send snapshots its buffer, records an event on the sender's stream and leaves (snapshot, event) in a mailbox; a receive blocks the
    receiving host thread until the message is there, makes its stream wait for the event and copies.  Only
    stream-ordered dependencies exist on the device (no kernel waits for another), so this is safe on one GPU."""

    class P2POp:
        def __init__(self, fn, tensor, peer, tag=0):
            self.fn, self.tensor, self.peer, self.tag = fn, tensor, peer, tag

    class _Work:
        def __init__(self, fn):
            self._fn = fn

        def wait(self):
            self._fn()

    def __init__(self, torch, world):
        import collections
        import threading

        self.torch, self.world = torch, world
        self.box = collections.defaultdict(list)
        self.cv = threading.Condition()
        self.local = threading.local()

    def isend(self, *a, **k):  # markers only: batch_isend_irecv looks at op.fn
        raise NotImplementedError

    def irecv(self, *a, **k):
        raise NotImplementedError

    def batch_isend_irecv(self, ops):
        torch, me = self.torch, self.local.rank
        works = []
        for op in ops:
            if op.fn == self.isend:
                # a real send has read its buffer when its work has been waited for; here the work is a no-op, so the
                # message is a snapshot taken in stream order (the sender may repack the buffer for its next application
                # before the receiving thread gets to copy)
                snap = op.tensor.clone()
                ev = torch.cuda.Event()
                ev.record(torch.cuda.current_stream())
                with self.cv:
                    self.box[(me, op.peer, op.tag)].append((snap, ev))
                    self.cv.notify_all()
                works.append(self._Work(lambda: None))
            else:
                stream = torch.cuda.current_stream()

                def recv(op=op, stream=stream):
                    with self.cv:
                        self.cv.wait_for(lambda: self.box[(op.peer, me, op.tag)], timeout=60)
                        src, ev = self.box[(op.peer, me, op.tag)].pop(0)
                    with torch.cuda.stream(stream):
                        stream.wait_event(ev)
                        op.tensor.copy_(src)

                works.append(self._Work(recv))
        return works


@pytest.mark.parametrize("gdims,grid", [((8, 8, 8, 16), (2, 1, 1, 1)), ((8, 8, 8, 16), (2, 2, 1, 1))])
def test_distributed_operator_with_in_process_ranks(torch, gdims, grid):
    """dd.DistributedOperator — the class bench.py --gpus N drives — with its ranks as threads of one process and
    torch.distributed replaced by `_InProcessDist`: pack, exchange on the side stream, interior, exterior, three
    applications in a row (buffers are reused), against the oracle on the global lattice."""
    import threading

    from paper_2407_00041_b200 import dd as wdd
    from paper_2407_00041_b200.decomp import Decomposition

    m0, csw = -0.4, 1.0
    d = Decomposition(gdims, grid)
    U = wdinputs.gauge_haar(gdims, 841)
    C = oracle.build_clover(gdims, m0, csw, U)
    psis = [wdinputs.spinor(gdims, 842 + k) for k in range(3)]
    refs = [oracle.apply(gdims, m0, U, C, p) for p in psis]
    fake = _InProcessDist(torch, d.world_size)
    outs = [[None] * d.world_size for _ in psis]
    errors = []

    def rank_main(r):
        try:
            fake.local.rank = r
            torch.cuda.set_device(0)
            with torch.cuda.stream(torch.cuda.Stream()):
                lo = wdd.LocalOperator(torch, d, r, m0, csw, d.extract(U, r), d.extract(C, r))
                op = wdd.DistributedOperator(torch, fake, lo)
                fake.P2POp  # noqa: B018  (the plan builder uses dist.P2POp / dist.isend / dist.irecv)
                for k, psi in enumerate(psis):
                    din, dout = lo.spinor(), lo.spinor()
                    dout.fill_(float("nan"))
                    wd.wd_pack_spinor(lo.h, din, np.ascontiguousarray(d.extract(psi[0], r)[None]), 1)
                    op.apply(dout, din, 1)
                    wd.wd_synchronize(lo.h)
                    loc = np.empty((1, int(np.prod(d.local_dims)), 12, 2))
                    wd.wd_unpack_spinor(lo.h, loc, dout, 1)
                    outs[k][r] = loc[0]
                lo.close()
        except Exception as exc:  # surfaced in the main thread
            errors.append((r, repr(exc)))

    threads = [threading.Thread(target=rank_main, args=(r,)) for r in range(d.world_size)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=180)
    assert not errors, errors
    for k, ref in enumerate(refs):
        out = np.empty_like(ref)
        for r in range(d.world_size):
            d.insert(out[0], r, outs[k][r])
        assert rel_l2(out, ref) <= TOL, k
