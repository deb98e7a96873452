"""Host logic of the domain decomposition on the CPU: rank-grid arithmetic, face enumeration, the order of the
point-to-point exchange, and the exchange itself over torch.distributed with the gloo backend (world size 2).
No operator arithmetic runs here — the payload of the exchange is the global site index of every face site, so that
the receiver can check that what arrived belongs to the site across the seam."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest

from paper_2407_00041_b200.decomp import Decomposition, default_grid
from paper_2407_00041_b200.dd import p2p_plan

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_default_grid_splits_t_then_z():
    g = (64, 64, 64, 64)
    assert [default_grid(n, g) for n in (1, 2, 4, 8, 16)] == [(1, 1, 1, 1), (2, 1, 1, 1), (4, 1, 1, 1), (4, 2, 1, 1), (4, 4, 1, 1)]
    with pytest.raises(ValueError):
        default_grid(3, g)
    with pytest.raises(ValueError):
        Decomposition((8, 8, 8, 8), (3, 1, 1, 1))


@pytest.mark.parametrize("gdims,grid", [((8, 8, 8, 8), (2, 1, 1, 1)), ((8, 12, 4, 6), (2, 3, 1, 2)), ((16, 8, 4, 4), (4, 2, 1, 1))])
def test_partition_is_exact_and_neighbours_are_periodic(gdims, grid):
    d = Decomposition(gdims, grid)
    V = int(np.prod(gdims))
    seen = np.zeros(V, dtype=int)
    for r in range(d.world_size):
        assert d.rank(d.coords(r)) == r
        seen[d.global_sites(r)] += 1
        for mu in range(4):
            assert d.neighbour(d.neighbour(r, mu, +1), mu, -1) == r
            n = r
            for _ in range(grid[mu]):
                n = d.neighbour(n, mu, +1)
            assert n == r  # periodic seam
    assert (seen == 1).all()  # the local lattices do not overlap and cover L
    # extract / insert are inverse
    f = np.arange(V * 3, dtype=float).reshape(V, 3)
    g = np.zeros_like(f)
    for r in range(d.world_size):
        d.insert(g, r, d.extract(f, r))
    assert np.array_equal(f, g)


@pytest.mark.parametrize("gdims,grid", [((8, 8, 8, 8), (2, 1, 1, 1)), ((8, 12, 4, 6), (2, 3, 1, 2)), ((16, 8, 4, 4), (4, 2, 1, 1))])
def test_faces_meet_across_the_seam(gdims, grid):
    """Face site k of my HIGH face and face site k of the +mu neighbour's LOW face are nearest neighbours in mu."""
    d = Decomposition(gdims, grid)
    strides = [gdims[1] * gdims[2] * gdims[3], gdims[2] * gdims[3], gdims[3], 1]
    for r in range(d.world_size):
        for mu in d.decomposed:
            hi = d.face_global_sites(r, mu, True)
            lo = d.face_global_sites(d.neighbour(r, mu, +1), mu, False)
            assert hi.size == lo.size == int(np.prod(d.local_dims)) // d.local_dims[mu]
            c_hi = (hi // strides[mu]) % gdims[mu]
            c_lo = (lo // strides[mu]) % gdims[mu]
            assert ((c_hi + 1) % gdims[mu] == c_lo).all()
            assert np.array_equal(hi - c_hi * strides[mu], lo - c_lo * strides[mu])  # same transverse coordinates


@pytest.mark.parametrize("grid", [(2, 1, 1, 1), (2, 2, 1, 1), (4, 2, 1, 1), (1, 2, 2, 2)])
def test_p2p_plan_matches_in_posting_order(grid):
    """For every ordered pair of ranks the k-th send posted by the source and the k-th receive posted by the
    destination carry the same tag and pair send_minus -> recv_from_plus, send_plus -> recv_from_minus."""
    d = Decomposition(tuple(8 * g for g in grid), grid)
    plans = [p2p_plan(d, r) for r in range(d.world_size)]
    for src in range(d.world_size):
        for dst in range(d.world_size):
            sends = [(n, mu, tag) for k, n, mu, peer, tag in plans[src] if k == "send" and peer == dst]
            recvs = [(n, mu, tag) for k, n, mu, peer, tag in plans[dst] if k == "recv" and peer == src]
            assert len(sends) == len(recvs)
            for (sn, smu, stag), (rn, rmu, rtag) in zip(sends, recvs):
                assert stag == rtag and smu == rmu
                assert (sn, rn) in (("send_minus", "recv_from_plus"), ("send_plus", "recv_from_minus"))
                if sn == "send_minus":
                    assert d.neighbour(src, smu, -1) == dst
                else:
                    assert d.neighbour(src, smu, +1) == dst


WORKER = r'''
import os, sys, json
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
from paper_2407_00041_b200.decomp import Decomposition
from paper_2407_00041_b200.dd import exchange_distributed
dist.init_process_group("gloo")
r = dist.get_rank()
d = Decomposition({gdims!r}, {grid!r})
buf = {{}}
for mu in d.decomposed:
    lo, hi = d.face_global_sites(r, mu, False), d.face_global_sites(r, mu, True)
    buf[(mu, "send_minus")] = torch.from_numpy(lo.astype(np.float64))           # stands for lambda on my low face
    buf[(mu, "send_plus")] = torch.from_numpy(hi.astype(np.float64) + 0.5)      # stands for chi on my high face
    buf[(mu, "recv_from_plus")] = torch.full((hi.size,), -1.0, dtype=torch.float64)
    buf[(mu, "recv_from_minus")] = torch.full((lo.size,), -1.0, dtype=torch.float64)
for req in exchange_distributed(dist, d, r, buf):
    req.wait()
ok = True
for mu in d.decomposed:
    # what I received from +mu is lambda on the LOW face of that neighbour; from -mu: chi on ITS high face
    ok &= np.array_equal(buf[(mu, "recv_from_plus")].numpy(), d.face_global_sites(d.neighbour(r, mu, +1), mu, False).astype(float))
    ok &= np.array_equal(buf[(mu, "recv_from_minus")].numpy(), d.face_global_sites(d.neighbour(r, mu, -1), mu, True).astype(float) + 0.5)
open(os.path.join({out!r}, "rank%d.json" % r), "w").write(json.dumps({{"rank": r, "ok": bool(ok), "n": len(d.decomposed)}}))
dist.barrier()
dist.destroy_process_group()
'''


@pytest.mark.parametrize("gdims,grid", [((8, 4, 4, 6), (2, 1, 1, 1)), ((4, 8, 4, 6), (1, 2, 1, 1))])
def test_face_exchange_over_gloo_world2(tmp_path, gdims, grid):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT, out=str(tmp_path), gdims=gdims, grid=grid))
    import socket

    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), str(script)]
    r = subprocess.run(cmd, capture_output=True, text=True, env=env, timeout=300)
    assert r.returncode == 0, r.stderr[-3000:]
    for k in (0, 1):
        res = json.loads((tmp_path / ("rank%d.json" % k)).read_text())
        assert res["ok"] and res["n"] == 1


def test_site_list_generators_draw_a_rank_part_without_the_global_field():
    """bench.py --gpus N: every rank draws only its own sites (and the link halo of its clover term).  The site-list
    generators must give, bit for bit, the rows of the global field the full generators give."""
    import wdinputs

    dims = (4, 6, 2, 8)
    d = Decomposition(dims, (2, 3, 1, 1))
    for cfg in (dict(gauge=("haar", 77)), dict(gauge=("exp", 78, 0.4))):
        U = wdinputs.config_gauge(cfg, dims)
        for rank in (0, 4):
            for halo in (0, 1):
                sites = d.global_sites(rank, halo)
                assert np.array_equal(wdinputs.config_gauge_sites(cfg, sites), U[sites])
                assert np.array_equal(wdinputs.config_gauge_sites(cfg, sites), d.extract(U, rank, halo))
    psi = wdinputs.spinor(dims, 79, nrhs=3)
    sites = d.global_sites(5)
    assert np.array_equal(wdinputs.spinor_sites(79, sites, 3), psi[:, sites])
