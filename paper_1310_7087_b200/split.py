"""A lattice divided into parts, ONE PART PER PROCESS (one process per GPU, torch.distributed): host-side bookkeeping only.

PAPER.md:124-128 sec 4: the lattice is divided, in general into unequal parts, along one spatial direction; "divided lattice
simulation differs from a full lattice simulation only in necessity to carry out the exchanging values of boundary sites".
Every step of the path runs in the kernels of libqcd_b200.so (qcd_slab_* in include/qcd.h): the part's sub-step, the packing
of a boundary layer into a message buffer and its unpacking into the neighbour's halo layer.  This module decides WHO sends
WHAT to WHOM and WHEN, and moves the buffers with torch.distributed point-to-point calls (NCCL over NVLink between GPUs;
gloo in the CPU test).  The same schedule, in C++ and with direct peer-memory copies, drives the single-process
qcd_split_* calls.

Conventions (include/qcd.h): the split direction is D-2; a part owns the layers [offset, offset + extent) (both even); it
keeps a copy of the next part's first layer and of the previous part's last layer.  After the sub-step (parity, mu) only the
array (parity, mu) has changed, so exactly two layers per part travel: side 0 (first own layer) to the previous part, side 1
(last own layer) to the next part.
"""


def partition(extent, n_parts, weights=None):
    """[(offset, extent_k)] of the n_parts parts of a direction of `extent` sites: even extents >= 2 that add up to `extent`;
    proportional to `weights` (relative device speeds: "unequal parts ... to hide the difference in devices performances",
    PAPER.md:124), equal as far as even extents allow by default."""
    if extent % 2 or n_parts < 1 or 2 * n_parts > extent:
        raise ValueError("need an even extent and 1 <= n_parts <= extent / 2")
    pairs = extent // 2                                     # the unit is two layers
    w = [1.0] * n_parts if weights is None else [float(x) for x in weights]
    if len(w) != n_parts or min(w) <= 0:
        raise ValueError("weights: one positive number per part")
    tot = sum(w)
    share = [1 + int((pairs - n_parts) * x / tot) for x in w]                     # at least one pair each
    rest = pairs - sum(share)
    # hand the remaining pairs to the parts with the largest unmet share
    order = sorted(range(n_parts), key=lambda k: (share[k] - 1) - (pairs - n_parts) * w[k] / tot)
    for k in order[:rest]:
        share[k] += 1
    out, off = [], 0
    for k in range(n_parts):
        out.append((off, 2 * share[k]))
        off += 2 * share[k]
    assert off == extent
    return out


def neighbours(rank, world):
    """(previous, next) part on the periodic split direction"""
    return (rank - 1) % world, (rank + 1) % world


def halo_messages(rank, world):
    """The two messages a part sends after every sub-step, as (pack side, destination rank, unpack side at the destination):
    its first own layer is the previous part's copy of "the next part's first layer" (unpack side 1), its last own layer the
    next part's copy of "the previous part's last layer" (unpack side 0)."""
    prev, nxt = neighbours(rank, world)
    return [(0, prev, 1), (1, nxt, 0)]


def sweep_schedule(D, n_hb, n_or):
    """[(kind, hit, parity, mu)] of one sweep: passes outermost, then parity, then direction (readings R1, R2)"""
    return [(0 if s < n_hb else 1, s if s < n_hb else 0, p, mu) for s in range(n_hb + n_or) for p in (0, 1) for mu in range(D)]


def exchange(dist, rank, world, packed, recv_like):
    """Send packed[side] (side 0 / 1) to the previous / next part and receive the two layers meant for this part.
    Returns {unpack side: tensor}.  With one part the lattice is its own neighbour on both sides."""
    if world == 1:
        return {1: packed[0], 0: packed[1]}
    got = {0: recv_like(), 1: recv_like()}
    ops = []
    for side, dst, _ in halo_messages(rank, world):
        ops.append(dist.P2POp(dist.isend, packed[side], dst, tag=side))
    prev, nxt = neighbours(rank, world)
    # what arrives from the next part is its side 0 (-> my unpack side 1), from the previous part its side 1 (-> unpack side 0)
    ops.append(dist.P2POp(dist.irecv, got[1], nxt, tag=0))
    ops.append(dist.P2POp(dist.irecv, got[0], prev, tag=1))
    # with two parts both neighbours are the same rank: its sends (side 0, then side 1) meet the receives in the same order
    # (NCCL matches point-to-point calls between a pair of ranks in order; gloo also by tag)
    for req in dist.batch_isend_irecv(ops):
        req.wait()
    return got


class DistributedSplitLattice:
    """One part of a divided lattice in this process.  `part` implements the per-part operations -- on the GPU the
    qcd_slab_* calls (GpuPart below), in the CPU test an oracle-backed stand-in:
        part.substep(beta, kind, hit, parity, mu, field)     update the part's own sites
        part.pack(parity, mu, side) -> tensor                boundary layer of the (parity, mu) array as a message
        part.unpack(parity, mu, side, tensor)                message -> halo layer
        part.recv_like() -> tensor                           empty message buffer
        part.measure_sums(field) -> (plane sums, Polyakov sum)
    """

    def __init__(self, dims, part, dist, rank, world):
        self.dims, self.D = tuple(dims), len(dims)
        self.part, self.dist, self.rank, self.world = part, dist, rank, world
        self.sweep_counter = 0

    def refresh_halos(self, parity, mu):
        packed = {side: self.part.pack(parity, mu, side) for side in (0, 1)}
        got = exchange(self.dist, self.rank, self.world, packed, self.part.recv_like)
        for side in (0, 1):
            self.part.unpack(parity, mu, side, got[side])

    def refresh_all(self):
        """after the links of the parts were set as a whole (init, set_links): every array's halo layers"""
        for parity in (0, 1):
            for mu in range(self.D):
                self.refresh_halos(parity, mu)

    def substep(self, beta, kind, hit, parity, mu, field=None):
        self.part.substep(beta, kind, hit, parity, mu, field)
        self.refresh_halos(parity, mu)

    def sweep(self, beta, n_hb, n_or, field=None):
        for kind, hit, parity, mu in sweep_schedule(self.D, n_hb, n_or):
            self.substep(beta, kind, hit, parity, mu, field)
        self.sweep_counter += 1
        self.part.set_sweep_counter(self.sweep_counter)

    def measure(self, field=None):
        """(plaquette total, planes, Polyakov loop) of the whole lattice: the parts' sums added over the ranks"""
        import torch
        planes, poly = self.part.measure_sums(field)
        t = torch.tensor(list(planes) + [poly.real, poly.imag], dtype=torch.float64, device=self.part.reduce_device())
        if self.world > 1:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM)
        t = t.cpu().numpy()
        V = 1
        for d in self.dims:
            V *= d
        planes = t[:-2] / V
        Vs = V // self.dims[-1]
        return float(planes.mean()), planes, complex(t[-2] / Vs, t[-1] / Vs)


class GpuPart:
    """The part of this process on its GPU: a slab handle of libqcd_b200.so and two message buffers per direction of travel."""

    def __init__(self, q, dims, Nc, precision, flags, offset, extent, device):
        import torch
        self.q, self.torch, self.device = q, torch, torch.device(device)
        self.lat = q.Lattice(dims, Nc, precision, flags, device=device, slab=(offset, extent))
        self.nbytes = self.lat.qcd_slab_halo_bytes()

    def recv_like(self):
        return self.torch.empty(self.nbytes, dtype=self.torch.uint8, device=self.device)

    def reduce_device(self):
        return self.device

    def init(self, start, seed):
        self.lat.qcd_init(start, seed)

    def substep(self, beta, kind, hit, parity, mu, field=None):
        self.lat.qcd_debug_substep(beta, kind, hit, parity, mu, field)

    def pack(self, parity, mu, side):
        buf = self.recv_like()
        self.lat.qcd_slab_halo_pack(parity, mu, side, buf.data_ptr(), self.nbytes)
        return buf

    def unpack(self, parity, mu, side, tensor):
        self.lat.qcd_slab_halo_unpack(parity, mu, side, tensor.data_ptr(), self.nbytes)

    def measure_sums(self, field=None):
        return self.lat.qcd_slab_measure_sums(field)

    def set_sweep_counter(self, v):
        self.lat.qcd_set_sweep_counter(v)


class StreamedLattice:
    """A divided lattice whose parts live in pinned HOST memory and pass through ONE device buffer, part by part, in every
    sub-step: the paper's other use of the division -- "when one device's memory is not enough".  Host-side
    bookkeeping only; every step runs in the kernels of the slab handles (qcd_slab_*), all created over the same device
    buffer.  Per sub-step and part: upload the part (its internal layout), unpack the latest boundary layers of its
    neighbours (the messages stay on the device: two layers per array and part, each kept until the next one replaces it),
    update, pack its own two boundary layers of the array just written for the neighbours, and download ONLY that
    (parity, mu) array -- the one the sub-step wrote, 1 / (2 D) of the part.  Each sub-step moves 1 + 1 / (2 D) times the
    lattice over the host link, so this is two orders of magnitude slower than a resident lattice: it
    exists for lattices beyond the 180 GB of one B200, and is tested on small ones, where it must reproduce the undivided
    sweep bit for bit."""

    def __init__(self, q, dims, Nc, precision, flags=0, n_parts=2, extents=None, device="cuda:0"):
        import torch
        self.q, self.torch, self.device = q, torch, torch.device(device)
        self.dims, self.D = tuple(int(x) for x in dims), len(dims)
        sd = self.D - 2
        if extents is None:
            self.parts = partition(self.dims[sd], n_parts)
        else:
            off, self.parts = 0, []
            for e in extents:
                self.parts.append((off, int(e)))
                off += int(e)
            assert off == self.dims[sd]
        self.n = len(self.parts)
        import ctypes
        arr = (ctypes.c_int * self.D)(*self.dims)
        probe = [int(q.lib().qcd_slab_bytes(self.D, arr, int(Nc), int(precision), int(flags), o, e)) for o, e in self.parts]
        with torch.cuda.device(self.device):
            self.buf = torch.empty(max(probe), dtype=torch.uint8, device=self.device)
        self.lat = [q.Lattice(self.dims, Nc, precision, flags, device=device, slab=pe, mem=self.buf) for pe in self.parts]
        self.host = [torch.empty(L.nbytes, dtype=torch.uint8, pin_memory=True) for L in self.lat]
        self.hbytes = [L.qcd_slab_halo_bytes() for L in self.lat]
        self.pending = [dict() for _ in range(self.n)]       # per part: {(parity, mu, unpack side): latest message tensor}
        self.resident = None
        self.sweep_counter = 0
        self.bytes_moved = 0

    def close(self):
        for L in self.lat:
            L.close()

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # ---- residency
    def _upload(self, k):
        """part k into the device buffer, then the latest boundary layers of its neighbours for every array (the halo layers
        of the host copy are not kept up to date: only the array a sub-step wrote travels back)"""
        L = self.lat[k]
        self.buf[:L.nbytes].copy_(self.host[k], non_blocking=True)
        self.bytes_moved += L.nbytes
        self.resident = k
        for (parity, mu, side), msg in self.pending[k].items():
            L.qcd_slab_halo_unpack(parity, mu, side, msg.data_ptr(), self.hbytes[k])
        # (an unpack tells the handle that its arrays were written behind its back: no early loads in the next kernel)
        if len(self.pending[k]) != 4 * self.D:
            raise RuntimeError("a part must have received all its halo layers before its first turn (call refresh_all)")

    def _download(self, k, array=None):
        """the resident part k back to its host copy: all of it, or only the (parity, mu) array number `array` =
        parity * D + mu (the internal layout is 2 D equal arrays, one per parity and direction, back to back)"""
        L = self.lat[k]
        a = L.nbytes // (2 * self.D)
        lo, hi = (0, L.nbytes) if array is None else (array * a, (array + 1) * a)
        self.host[k][lo:hi].copy_(self.buf[lo:hi], non_blocking=True)
        self.torch.cuda.current_stream().synchronize()      # the buffer is reused by the next part
        self.bytes_moved += hi - lo

    def _post(self, k, parity, mu):
        """the two boundary layers of array (parity, mu) of the resident part k, as messages to its neighbours"""
        L = self.lat[k]
        for side, dst, uside in halo_messages(k, self.n):
            msg = self.torch.empty(self.hbytes[k], dtype=self.torch.uint8, device=self.device)
            L.qcd_slab_halo_pack(parity, mu, side, msg.data_ptr(), self.hbytes[k])
            self.pending[dst][(parity, mu, uside)] = msg

    def refresh_all(self):
        """after the parts were set as a whole: every array's boundary layers to the neighbours"""
        for k in range(self.n):
            L = self.lat[k]
            self.buf[:L.nbytes].copy_(self.host[k], non_blocking=True)
            for parity in (0, 1):
                for mu in range(self.D):
                    self._post(k, parity, mu)
            self.torch.cuda.current_stream().synchronize()

    # ---- the lattice as a whole
    def init(self, start, seed):
        for k, L in enumerate(self.lat):
            L.qcd_init(start, seed)
            self._download(k)
        self.refresh_all()

    def set_seed(self, seed):
        for L in self.lat:
            L.qcd_set_seed(seed)

    def set_links(self, links):
        """canonical [lex][mu][N][N] of the whole lattice"""
        import numpy as np
        sd = self.D - 2
        a = np.asarray(links).reshape(tuple(reversed(self.dims)) + np.asarray(links).shape[1:])
        for k, (off, ext) in enumerate(self.parts):
            idx = [slice(None)] * self.D
            idx[self.D - 1 - sd] = slice(off, off + ext)
            blk = np.ascontiguousarray(a[tuple(idx)])
            self.lat[k].qcd_set_links(blk.reshape((-1,) + blk.shape[self.D:]))
            self._download(k)
        self.refresh_all()

    def get_links(self):
        import numpy as np
        sd = self.D - 2
        out = None
        for k, (off, ext) in enumerate(self.parts):
            L = self.lat[k]
            self.buf[:L.nbytes].copy_(self.host[k], non_blocking=True)
            blk = L.qcd_get_links()
            if out is None:
                out = np.zeros(tuple(reversed(self.dims)) + blk.shape[1:], dtype=blk.dtype)
            idx = [slice(None)] * self.D
            idx[self.D - 1 - sd] = slice(off, off + ext)
            shape = list(reversed(self.dims))
            shape[self.D - 1 - sd] = ext
            out[tuple(idx)] = blk.reshape(tuple(shape) + blk.shape[1:])
        return out.reshape((-1,) + out.shape[self.D:])

    def substep(self, beta, kind, hit, parity, mu, field=None):
        for k in range(self.n):
            self._upload(k)
            self.lat[k].qcd_debug_substep(beta, kind, hit, parity, mu, field)
            self._post(k, parity, mu)
            self._download(k, parity * self.D + mu)

    def sweep(self, beta, n_hb, n_or, field=None):
        for kind, hit, parity, mu in sweep_schedule(self.D, n_hb, n_or):
            self.substep(beta, kind, hit, parity, mu, field)
        self.sweep_counter += 1
        for L in self.lat:
            L.qcd_set_sweep_counter(self.sweep_counter)

    def measure(self, field=None):
        import numpy as np
        planes, poly = None, 0j
        for k in range(self.n):
            L = self.lat[k]
            self.buf[:L.nbytes].copy_(self.host[k], non_blocking=True)
            for (parity, mu, side), msg in self.pending[k].items():
                L.qcd_slab_halo_unpack(parity, mu, side, msg.data_ptr(), self.hbytes[k])
            pk, lk = L.qcd_slab_measure_sums(field)
            planes = pk if planes is None else planes + pk
            poly += lk
        V = int(np.prod(self.dims))
        planes = planes / V
        Vs = V // self.dims[-1]
        return float(planes.mean()), planes, poly / Vs
