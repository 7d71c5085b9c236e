"""Run by tests/test_split_cpu.py under torch.distributed.run with 2 CPU ranks (gloo).  Each rank owns one part of a lattice
divided along direction D-2 and drives it with paper_1310_7087_b200/split.py (the same bookkeeping the GPU path uses); the
per-part operations are supplied by an ORACLE-backed stand-in for the GPU slab: the whole configuration is held as a numpy
array that is NaN everywhere except on the rank's own layers and its two halo layers; a sub-step hands that array to the
oracle, keeps the new values of the rank's own sites only, and the boundary layers travel through torch.distributed.  At the
end the parts are gathered and compared with the undivided oracle run."""
import importlib.util
import json
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import oracle  # noqa: E402
from tests import np_lattice as npl  # noqa: E402
from tests.inputs import random_links  # noqa: E402

spec = importlib.util.spec_from_file_location("qcd_split_host", os.path.join(ROOT, "paper_1310_7087_b200", "split.py"))
sp = importlib.util.module_from_spec(spec)
spec.loader.exec_module(sp)


class OraclePart:
    def __init__(self, dims, Nc, offset, extent, links, seed):
        self.dims, self.D, self.Nc = tuple(dims), len(dims), Nc
        self.sd = self.D - 2
        self.off, self.ext, self.L = offset, extent, dims[self.sd]
        self.V = int(np.prod(dims))
        self.par = npl.site_parity(dims)
        coords = np.stack(np.unravel_index(np.arange(self.V), dims[::-1]), axis=-1)[:, ::-1]
        self.layer = coords[:, self.sd]
        self.own = (self.layer >= offset) & (self.layer < offset + extent)
        self.halo_next = self.layer == (offset + extent) % self.L          # copy of the next part's first layer
        self.halo_prev = self.layer == (offset - 1) % self.L               # copy of the previous part's last layer
        self.state = np.full((self.V, self.D, Nc, Nc), np.nan + 0j, dtype=np.complex128)
        self.state[self.own] = links[self.own]                              # halos arrive by refresh_all()
        self.O = oracle.OracleLattice(dims, Nc)
        self.O.set_seed(seed)
        self.sent = 0

    def substep(self, beta, kind, hit, parity, mu, field=None):
        self.O.set_links(self.state)
        self.O.substep(beta, kind, hit, parity, mu, field)
        new = self.O.get_links()
        upd = self.own & (self.par == parity)
        self.state[upd, mu] = new[upd, mu]

    def _layer_sites(self, which, parity):
        return np.flatnonzero(which & (self.par == parity))

    def pack(self, parity, mu, side):
        lay = self.off if side == 0 else self.off + self.ext - 1
        self.sent += 1
        return torch.from_numpy(np.ascontiguousarray(self.state[self._layer_sites(self.layer == lay, parity), mu]))

    def unpack(self, parity, mu, side, tensor):
        which = self.halo_prev if side == 0 else self.halo_next
        self.state[self._layer_sites(which, parity), mu] = tensor.numpy()

    def recv_like(self):
        n = self.V // self.L // 2
        return torch.empty((n, self.Nc, self.Nc), dtype=torch.complex128)

    def reduce_device(self):
        return "cpu"

    def set_sweep_counter(self, v):
        self.O.sweep_counter = v

    def measure_sums(self, field=None):
        # plaquettes based at own sites reach one layer forward (the "next" halo); Polyakov lines are local
        g = npl.to_grid(self.state, self.dims)
        N = self.Nc
        sums = []
        own_g = self.own.reshape(tuple(reversed(self.dims)))
        for mu in range(self.D):
            for nu in range(mu + 1, self.D):
                Um, Un = g[..., mu, :, :], g[..., nu, :, :]
                P = Um @ npl.shift(Un, self.dims, mu) @ npl.dag(npl.shift(Um, self.dims, nu)) @ npl.dag(Un)
                t = np.trace(P, axis1=-2, axis2=-1).real / N
                sums.append(float(t[own_g].sum()))
        gt = g[..., self.D - 1, :, :]
        P = gt[0]
        for t in range(1, self.dims[self.D - 1]):
            P = P @ gt[t]
        tr = np.trace(P, axis1=-2, axis2=-1) / N
        return np.array(sums), complex(tr[own_g[0]].sum())


def main():
    case = sys.argv[1]
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    if case == "su3_4d":
        dims, Nc, beta, weights, n_hb, n_or = (4, 4, 8, 4), 3, 5.7, None, 1, 1
    else:
        dims, Nc, beta, weights, n_hb, n_or = (6, 12, 4), 2, 2.5, [1, 2], 1, 2
    D = len(dims)
    links = random_links(dims, Nc, 41, 0.35)
    parts = sp.partition(dims[D - 2], world, weights)
    off, ext = parts[rank]
    part = OraclePart(dims, Nc, off, ext, links, seed=77)
    lat = sp.DistributedSplitLattice(dims, part, dist, rank, world)
    lat.refresh_all()
    n_refresh = part.sent
    lat.sweep(beta, n_hb, n_or)
    n_sub = 2 * D * (n_hb + n_or)
    per_substep = (part.sent - n_refresh) // n_sub
    lat.sweep(beta, n_hb, n_or)
    tot, planes, poly = lat.measure()
    # gather the parts
    mine = np.where(part.own[:, None, None, None], part.state, 0.0)
    nan_free = bool(np.isfinite(part.state[part.own].view(np.float64)).all())
    t = torch.from_numpy(np.ascontiguousarray(mine).view(np.float64))
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    full = t.numpy().view(np.complex128).reshape(mine.shape)
    # the undivided oracle
    O = oracle.OracleLattice(dims, Nc)
    O.set_links(links)
    O.set_seed(77)
    O.sweep(beta, n_hb, n_or)
    O.sweep(beta, n_hb, n_or)
    ref = O.get_links()
    tot_o, planes_o, poly_o = O.measure()
    out = {"parts": parts, "split_extent": dims[D - 2], "links_equal": bool(np.array_equal(full, ref)), "nan_free_owned": nan_free,
           "max_measure_diff": float(max(np.max(np.abs(planes - planes_o)), abs(poly - poly_o), abs(tot - tot_o))),
           "messages_per_substep_per_rank": per_substep}
    flags = torch.tensor([1.0 if out["links_equal"] and nan_free else 0.0])
    dist.all_reduce(flags, op=dist.ReduceOp.MIN)
    out["links_equal"] = out["links_equal"] and bool(flags.item() == 1.0)
    dist.barrier()
    dist.destroy_process_group()
    if rank == 0:
        print("SPLIT " + json.dumps(out), flush=True)


if __name__ == "__main__":
    main()
