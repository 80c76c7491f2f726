"""Multi-GPU Cshift and shifted product on x3 slabs (PAPER.md P:219 names Cshift as the
operation after the site-local product).  The site-local path shards with no exchange; a shift along x3 is the one
operation that needs the neighbour's planes.  This module executes shard.cshift_plan:

    pack my face (su3_face_pack)  ->  send/recv (torch.distributed P2P: NCCL over NVLink)  ||  local shift of the bulk
    (su3_cshift / su3_mul_shift on the rank's own slab, the full-bandwidth kernels)  ->  unpack the received face
    (su3_face_unpack) over the planes the local periodic shift filled from the wrong side.

The face is 1/l3 of the slab per unit of displacement, so the transfer hides behind the local kernel.  The packed
face is a scalar-layout field of nface planes whatever the layout of the slab, so ranks exchange it blindly and the
shifted product fixes its face with the ordinary su3_mul on packed buffers (bit-identical FMA chain).
Argument marshalling and sequencing only: every byte is moved by the library's kernels or by the collective.
`comm` abstracts the exchange so that a single process can stand in for several ranks (LoopbackComm; 1-GPU tests);
`ops` abstracts the kernels so that the sequencing can be driven on CPU under gloo with a checker's kernels
(tests/test_halo_gloo.py); the product path is DistComm + CudaOps, and nothing else is ever the default."""
from . import shard


class DistComm:
    """torch.distributed point-to-point exchange (backend nccl: device tensors; transfers run on NCCL's own stream
    concurrently with kernels issued afterwards on the current stream; wait() orders the current stream after them)."""

    def __init__(self, dist):
        self.dist = dist
        self.rank, self.world = dist.get_rank(), dist.get_world_size()

    def exchange(self, send, to, recv, frm):
        """send tensor -> rank `to`, recv tensor <- rank `frm`; returns a list of objects with wait()"""
        d = self.dist
        if to == self.rank and frm == self.rank:
            recv.copy_(send)
            return []
        return d.batch_isend_irecv([d.P2POp(d.isend, send, to), d.P2POp(d.irecv, recv, frm)])


class LoopbackComm:
    """All `world` ranks live in ONE process on one GPU (tests, 1-GPU functional checks): a send is kept in a mailbox
    until the receiving rank waits.  Every rank must issue its exchanges (SlabShift.start) before any rank finishes."""

    def __init__(self, world):
        self.world = world
        self.mail = {}

    def for_rank(self, rank):
        return _LoopbackRank(self, rank)


class _LoopbackRank:
    def __init__(self, hub, rank):
        self.hub, self.rank, self.world = hub, rank, hub.world

    def exchange(self, send, to, recv, frm):
        self.hub.mail.setdefault((self.rank, to), []).append(send)
        return [_LoopbackWait(self.hub, frm, self.rank, recv)]


class _LoopbackWait:
    def __init__(self, hub, frm, to, recv):
        self.hub, self.key, self.recv = hub, (frm, to), recv

    def wait(self):
        self.recv.copy_(self.hub.mail[self.key].pop(0))


class CudaOps:
    """The product's kernels: libsu3stream through the binding.  Fields are su3.Field objects."""

    def __init__(self):
        import torch
        import paper_1710_09409_b200 as su3
        self.su3, self.torch = su3, torch

    def l3(self, f):
        return f.desc.L[shard.SLAB_DIM]

    def key(self, f):
        d = f.desc
        return (f.kind, tuple(d.L), d.n_lorentz, d.prec, str(f.tensor.device))

    def face_buffer(self, f, n):
        nb = self.su3.su3_face_bytes(f, shard.SLAB_DIM, n)
        return self.torch.empty(nb, dtype=self.torch.uint8, device=f.tensor.device)

    def slab_like(self, f):
        return self.su3.Field(f.desc, self.torch.empty(f.nbytes, dtype=self.torch.uint8, device=f.tensor.device), kind=f.kind)

    def payload(self, f):
        return f.tensor

    def face_pack(self, buf, x, plane0, n):
        self.su3.su3_face_pack(buf, x, shard.SLAB_DIM, plane0, n)

    def face_unpack(self, z, buf, plane0, n):
        self.su3.su3_face_unpack(z, buf, shard.SLAB_DIM, plane0, n)

    def cshift(self, z, y, dim, disp):
        self.su3.su3_cshift(z, y, dim, disp)

    def mul_shift(self, z, x, y, dim, disp):
        self.su3.su3_mul_shift(z, x, y, dim, disp)

    def copy(self, z, y):
        self.su3.su3_copy(z, y)

    def mul(self, z, x, y):
        self.su3.su3_mul(z, x, y)

    def face_mul(self, zb, xb, hb, like, n):
        """zb = xb . hb on packed faces: they ARE scalar-layout fields of n planes (include/su3stream.h)"""
        su3 = self.su3
        L = tuple(like.desc.L)
        d = su3.make_desc((L[0], L[1], L[2], n), n_lorentz=like.desc.n_lorentz, prec=like.desc.prec)
        fz, fx, fh = (su3.su3_field_wrap(d, t) for t in (zb, xb, hb))
        su3.su3_mul(fz, fx, fh)


class SlabShift:
    """Cshift / shifted product along any dimension for one rank's slab.  Buffers for the faces (and, for shifts by a
    whole slab or more, one scratch slab) are allocated once per size and reused.

    Because the buffers are shared by every shift of same-shaped fields, only ONE exchanging shift per field shape may
    be between start() and its finish_*(): a second start() would overwrite the send buffer while the first send may
    still be running, and the receive buffer before the first unpack.  start() raises RuntimeError in that case instead
    of corrupting the first shift; finish the first one (or use a second SlabShift object, which has its own buffers).
    Shifts that need no exchange (another dimension, or one rank) are not restricted."""

    def __init__(self, comm, ops=None):
        self.comm = comm
        self.ops = ops if ops is not None else CudaOps()
        self._buf = {}
        self._in_flight = set()

    def _cached(self, key, make):
        if key not in self._buf:
            self._buf[key] = make()
        return self._buf[key]

    def start(self, y, dim, disp):
        """Phase 1 (every rank, before any rank calls finish_*): issue the sends/receives a shift of `y` needs."""
        c, o = self.comm, self.ops
        if dim != shard.SLAB_DIM or c.world == 1:
            return {"local": True, "dim": dim, "disp": disp, "y": y}
        plan = shard.cshift_plan(o.l3(y), c.rank, c.world, disp)
        if o.key(y) in self._in_flight:
            raise RuntimeError("SlabShift: a shift of a field of this shape is still between start() and finish_*(); "
                               "its face buffers are shared -- finish it first, or use another SlabShift object")
        self._in_flight.add(o.key(y))
        st = {"local": False, "plan": plan, "src": y, "works": [], "bulk_works": [], "key": o.key(y)}
        n = plan["nface"]
        if n:
            sbuf = self._cached(("send", n, o.key(y)), lambda: o.face_buffer(y, n))
            rbuf = self._cached(("recv", n, o.key(y)), lambda: o.face_buffer(y, n))
            o.face_pack(sbuf, y, plan["send_plane0"], n)
            st["works"] += c.exchange(sbuf, plan["face_to"], rbuf, plan["face_from"])
            st["halo"] = rbuf
        if plan["bulk_from"] != c.rank:
            scr = self._cached(("slab", o.key(y)), lambda: o.slab_like(y))
            st["bulk_works"] += c.exchange(o.payload(y), plan["bulk_to"], o.payload(scr), plan["bulk_from"])
            st["src"] = scr
        return st

    def finish_cshift(self, z, st):
        """Phase 2: z[s] = y[s + disp*dim_hat] on the GLOBAL lattice (the local kernel overlaps the face transfer)."""
        o = self.ops
        if st["local"]:
            o.cshift(z, st["y"], st["dim"], st["disp"])
            return
        plan = st["plan"]
        for w in st["bulk_works"]:
            w.wait()
        if plan["shift"]:
            o.cshift(z, st["src"], shard.SLAB_DIM, plan["shift"])
        else:
            o.copy(z, st["src"])
        for w in st["works"]:
            w.wait()
        if plan["nface"]:
            o.face_unpack(z, st["halo"], plan["dst_plane0"], plan["nface"])
        self._in_flight.discard(st["key"])

    def finish_mul_shift(self, z, x, st):
        """Phase 2: z[s] = x[s] . y[s + disp*dim_hat] on the GLOBAL lattice.  The bulk is one su3_mul_shift (or su3_mul)
        on the slab; the face is x's planes times the received planes, by su3_mul on the packed (scalar-layout) faces.
        z may be x (su3stream.h allows it for the product): x's face planes are packed BEFORE the bulk kernel runs,
        because with z = x that kernel overwrites them with products of the wrongly wrapped planes."""
        o = self.ops
        if st["local"]:
            o.mul_shift(z, x, st["y"], st["dim"], st["disp"])
            return
        plan = st["plan"]
        n = plan["nface"]
        if n:
            xb = self._cached(("xface", n, o.key(x)), lambda: o.face_buffer(x, n))
            o.face_pack(xb, x, plan["dst_plane0"], n)
        for w in st["bulk_works"]:
            w.wait()
        if plan["shift"]:
            o.mul_shift(z, x, st["src"], shard.SLAB_DIM, plan["shift"])
        else:
            o.mul(z, x, st["src"])
        for w in st["works"]:
            w.wait()
        if n:
            zb = self._cached(("zface", n, o.key(x)), lambda: o.face_buffer(x, n))
            o.face_mul(zb, xb, st["halo"], x, n)
            o.face_unpack(z, zb, plan["dst_plane0"], n)
        self._in_flight.discard(st["key"])

    def cshift(self, z, y, dim, disp):
        self.finish_cshift(z, self.start(y, dim, disp))

    def mul_shift(self, z, x, y, dim, disp):
        self.finish_mul_shift(z, x, self.start(y, dim, disp))


class PeerShift:
    """The same shifts when the neighbouring slabs are MAPPED into this process (peer memory over NVLink: CUDA IPC or
    symmetric memory give a device pointer that su3_field_wrap takes like any other; in the 1-GPU tests the
    "neighbours" are simply other fields on the same device).  No staging buffer and no collective call: the kernels
    read the neighbour's planes themselves.  |disp| must be below the slab's extent; both neighbours are passed and
    the sign of disp picks one."""

    def __init__(self):
        import torch
        import paper_1710_09409_b200 as su3
        self.su3, self.torch = su3, torch
        self._buf = {}

    def cshift(self, z, y, y_next, y_prev, disp):
        """z[s] = Y[s + disp*e3], one kernel (su3_cshift_slab) unless x3 is split over virtual nodes (then two)."""
        self.su3.su3_cshift_slab(z, y, y_next if disp > 0 else y_prev, disp)

    def mul_shift(self, z, x, y, y_next, y_prev, disp):
        """z[s] = x[s] . Y[s + disp*e3]: the periodic product on the slab, then the |disp| wrapped planes again as
        su3_mul on packed faces -- x's planes times the neighbour's planes, packed straight out of its memory.
        z may be x: x's face is packed before the bulk kernel overwrites those planes."""
        su3 = self.su3
        n = abs(disp)
        l3 = x.desc.L[shard.SLAB_DIM]
        if n >= l3:                                                # checked before anything is launched
            raise ValueError("|disp| = %d must be below the slab's %d planes" % (n, l3))
        if n == 0:
            su3.su3_mul_shift(z, x, y, shard.SLAB_DIM, 0)
            return
        nbr = y_next if disp > 0 else y_prev
        dst0, src0 = (l3 - n, 0) if disp > 0 else (0, l3 - n)
        nb = su3.su3_face_bytes(x, shard.SLAB_DIM, n)
        key = (nb, str(x.tensor.device))
        if key not in self._buf:
            self._buf[key] = [self.torch.empty(nb, dtype=self.torch.uint8, device=x.tensor.device) for _ in range(3)]
        xb, hb, zb = self._buf[key]
        su3.su3_face_pack(xb, x, shard.SLAB_DIM, dst0, n)
        su3.su3_mul_shift(z, x, y, shard.SLAB_DIM, disp)
        su3.su3_face_pack(hb, nbr, shard.SLAB_DIM, src0, n)
        L = tuple(x.desc.L)
        d = su3.make_desc((L[0], L[1], L[2], n), n_lorentz=x.desc.n_lorentz, prec=x.desc.prec)
        fz, fx, fh = (su3.su3_field_wrap(d, t) for t in (zb, xb, hb))
        su3.su3_mul(fz, fx, fh)
        su3.su3_face_unpack(z, zb, shard.SLAB_DIM, dst0, n)
