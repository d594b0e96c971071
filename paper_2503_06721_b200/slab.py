"""Host logic of the sharded operator: t-direction block partition and the face exchange.

One process per GPU; rank r owns the global time slices [t_start, t_start + T_loc) (Fig 1).  Per operator
application one exchange step of PROJECTED half-spinor faces (L624): the first owned slice goes to the previous rank, the last
to the next one, point to point (torch.distributed isend / irecv: NCCL over NVLink on GPUs, gloo on CPU in the tests).  No
arithmetic here: packing, unpacking and the operator are the library's kernels (hirep_halo_pack / hirep_halo_unpack /
hirep_set_region in include/hirep_b200.h).  Unmeasured on multi-GPU hardware this round.
"""
from __future__ import annotations


def partition(T_glob: int, world: int):
    """[(t_start, T_loc)] per rank: contiguous blocks of an even number of slices, as equal as possible, even offsets."""
    if T_glob % 2 or world < 1 or T_glob < 2 * world:
        raise ValueError("T_glob=%d cannot be split into %d slabs of an even number (>= 2) of slices" % (T_glob, world))
    pairs = T_glob // 2                     # distribute PAIRS of slices so that every T_loc and t_start is even
    base, extra = divmod(pairs, world)
    out, t = [], 0
    for r in range(world):
        n = 2 * (base + (1 if r < extra else 0))
        out.append((t, n))
        t += n
    return out


def neighbours(rank: int, world: int):
    """(previous, next) rank in t, periodic: the boundary condition lives in the links of the owning rank."""
    return (rank - 1) % world, (rank + 1) % world


def exchange_faces(dist, rank: int, world: int, face_first, face_last, recv_from_next, recv_from_prev):
    """Send the first owned slice's face to the previous rank and the last one's to the next; receive the next rank's first
    face into recv_from_next (it fills this rank's LAST ghost slice) and the previous rank's last face into recv_from_prev
    (ghost slice 0).  All four are contiguous tensors of hirep_halo_bytes bytes.  world == 1: the slab wraps onto itself."""
    if world == 1:
        recv_from_next.copy_(face_first)
        recv_from_prev.copy_(face_last)
        return
    prev, nxt = neighbours(rank, world)
    reqs = [dist.isend(face_first, prev, tag=0), dist.isend(face_last, nxt, tag=1),
            dist.irecv(recv_from_next, nxt, tag=0), dist.irecv(recv_from_prev, prev, tag=1)]
    for q in reqs:
        q.wait()


def apply_sharded(geom, dist, rank, world, op, in_half_or_full, halves, stream_sync=None):
    """One sharded application with the inner/boundary split of Fig 1: pack faces, start the exchange, run the INTERIOR,
    complete the exchange, unpack into the ghost slices, run the BOUNDARY slabs.  `halves`: the native half-lattice views of the
    input whose faces the operator reads (one for Dphi_eo / Dphi_oe, two for Dphi); `op(region)` launches the operator."""
    from . import hirep
    packed = [(geom.halo_pack(0, h), geom.halo_pack(1, h)) for h in halves]
    recv = [(geom._buf(p[0].numel()), geom._buf(p[1].numel())) for p in packed]
    if stream_sync is not None:
        stream_sync()                       # the packed faces are complete before the transport reads them
    geom.set_region(hirep.REGION_INTERIOR)
    op()
    for (f0, f1), (rn, rp) in zip(packed, recv):
        exchange_faces(dist, rank, world, f0, f1, rn, rp)
    for h, (rn, rp) in zip(halves, recv):
        geom.halo_unpack(0, h, rn)          # next rank's first slice -> last ghost slice
        geom.halo_unpack(1, h, rp)          # previous rank's last slice -> ghost slice 0
    geom.set_region(hirep.REGION_BOUNDARY)
    op()
    geom.set_region(hirep.REGION_OWNED)
