"""Host logic of the sharded evaluation (paper_2111_11473_b200/sharded.py) on CPU ranks: world_size 2 and 3 over gloo.

The CUDA kernels cannot run here, so each rank is played by a backend built on the dense oracle that follows the same
protocol: partial sums over the rank's Cholesky range (thc_shard_range, from the C library) and its
row block of the T2^2 terms -> one all-reduce -> redundant finish (Alg.9 from the summed xi).  The test checks that
ranges, the reduction and the finish step reproduce the unsharded oracle.  The CUDA backend itself is checked against
the unsharded CUDA path in test_gpu_sharded.py (ranks emulated one after the other on one device).
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from conftest import small_inputs


class OracleBackend:
    def __init__(self, x):
        from oracle import dense
        self.x, self.dense = x, dense
        self.t = dense.expand_t(x.Xo, x.Xv, x.Z)
        self.thc = dense.thc_ovov(x.Y[:x.o], x.Y[x.o:], x.V)

    def _ranges(self, rank, world):
        import paper_2111_11473_b200 as thc
        return thc.thc_shard_range(self.x.NL, self.x.NP, rank, world)

    def shard(self, rank, world):
        x, d = self.x, self.dense
        L0, L1, P0, P1 = self._ranges(rank, world)
        NP, o, v = x.NP, x.o, x.v
        cd = d.cd_eris(x.B_oo[L0:L1], x.B_ov[L0:L1], x.B_vv[L0:L1])          # ERIs of this rank's Cholesky range
        om = d.omega_terms(self.t, cd, self.thc, np.zeros(o), np.zeros(v))
        lin = sum(d.project(x.Xo, x.Xv, om[k]) for k in ("s1", "s2", "s3"))   # bilinear in B: additive over ranges
        quad = np.zeros((NP, NP))
        quad[P0:P1] = (d.project(x.Xo, x.Xv, om["s6"]) + d.project(x.Xo, x.Xv, om["s7"]))[P0:P1]
        return torch.from_numpy(np.concatenate([lin.ravel(), quad.ravel(), om["xi_oo"].ravel(), om["xi_vv"].ravel()]))

    def finish(self, packed):
        x, d = self.x, self.dense
        NP, o, v = x.NP, x.o, x.v
        p = packed.numpy()
        lin, quad = p[:NP * NP].reshape(NP, NP), p[NP * NP:2 * NP * NP].reshape(NP, NP)
        xi_oo = p[2 * NP * NP:2 * NP * NP + o * o].reshape(o, o)
        xi_vv = p[2 * NP * NP + o * o:].reshape(v, v)
        t = self.t
        Foo, Fvv = np.diag(x.eps[:o]) + xi_oo, np.diag(x.eps[o:]) + xi_vv     # Alg.9 lines 5-6 with the summed xi
        s9 = (np.einsum("iajc,bc->iajb", t, Fvv) + np.einsum("icjb,ac->iajb", t, Fvv)
              - np.einsum("iakb,kj->iajb", t, Foo) - np.einsum("kajb,ki->iajb", t, Foo))
        return torch.from_numpy(lin + quad + d.project(x.Xo, x.Xv, s9))

    def energy_shard(self, rank, world):
        L0, L1, _, _ = self._ranges(rank, world)
        B = self.x.B_ov[L0:L1]
        return torch.tensor([self.dense.energy_from(self.t, np.einsum("Lia,Ljb->iajb", B, B))], dtype=torch.float64)


def _worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2111_11473_b200.sharded import residual_sharded, energy_sharded
    x = small_inputs(4, 7, 11, 10, 13, seed=6, zmul=30.0)
    be = OracleBackend(x)
    R = residual_sharded(be).numpy()
    E = float(energy_sharded(be)[0])
    np.save(os.path.join(out_dir, f"R{rank}.npy"), R)
    np.save(os.path.join(out_dir, f"E{rank}.npy"), np.array([E]))
    dist.destroy_process_group()


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


@pytest.mark.parametrize("world", [2, 3])
def test_sharded_residual_over_gloo(world, tmp_path):
    from oracle import dense
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    x = small_inputs(4, 7, 11, 10, 13, seed=6, zmul=30.0)
    ref = dense.residual_and_energy(x.Xo, x.Xv, x.Z, x.B_ov, x.B_oo, x.B_vv, x.Y, x.V, x.eps)
    for r in range(world):
        R = np.load(tmp_path / f"R{r}.npy")
        E = np.load(tmp_path / f"E{r}.npy")[0]
        assert np.abs(R - ref["R"]).max() <= 1e-12 * np.abs(ref["R"]).max(), r
        assert abs(E - ref["E"]) <= 1e-12 * max(1.0, abs(ref["E"]))


def test_shard_ranges_partition():
    import paper_2111_11473_b200 as thc
    for NL, NP, world in [(60, 50, 1), (360, 300, 8), (7, 5, 8), (7500, 5000, 3)]:
        Ls, Ps = [], []
        for r in range(world):
            L0, L1, P0, P1 = thc.thc_shard_range(NL, NP, r, world)
            Ls.append((L0, L1)); Ps.append((P0, P1))
        for rng, n in ((Ls, NL), (Ps, NP)):
            assert rng[0][0] == 0 and rng[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(rng, rng[1:]))
            sizes = [b - a for a, b in rng]
            assert max(sizes) - min(sizes) <= 1
