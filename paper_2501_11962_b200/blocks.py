"""Bead-block sharding of a path over ranks: the paper's parallel layout.

The paper runs one bead per processing element and exchanges data between the owners of ADJACENT beads only, with
non-blocking point-to-point messages; its weak-scaling experiment grows the path with the machine
(PAPER.md:147-157).  Here every rank (one process, one GPU) owns a contiguous block of beads and a bead-block context
(`binding.Mop(..., block=(first, n_path))`, mop.h "bead-block mode").  One evaluation of V_eff and its gradient:

    1. halo:   every rank sends its first bead R^{n0} to the left neighbour and receives R^{n1} from the right one
    2. pass 1: mop_block_pass1 (lists, forces, eta; writes K eta of the block's last bead)
    3. halo:   that K eta goes to the right neighbour, the left neighbour's arrives    } these two overlap: the
    4. pass 2: mop_block_pass2 (H.eta)                                                  } transfer is asynchronous
    5. assembly: mop_block_assemble with the left halo; V_eff = all-reduce(sum) of the per-block values (8 bytes)

Per evaluation and block edge: Q x 12 bytes each way (1.8 MB at 150,000 atoms).  The module only moves tensors with
`torch.distributed` point-to-point operations (NCCL for CUDA tensors, gloo for CPU tensors: the same code), all of the
arithmetic is in the library.  `engine` is anything with the three block calls of `binding.Mop`.
"""
import torch
import torch.distributed as dist


def partition(n_beads_path, world):
    """Contiguous blocks, sizes differing by at most one: [(first_bead, n_beads)] per rank.  Every rank gets >= 1 bead."""
    if world < 1 or n_beads_path < world:
        raise ValueError("need 1 <= world <= n_beads_path (every rank owns at least one bead)")
    base, extra = divmod(n_beads_path, world)
    out, first = [], 0
    for r in range(world):
        n = base + (1 if r < extra else 0)
        out.append((first, n))
        first += n
    return out


def _exchange(send_to, send_tensor, recv_from, recv_tensor, group=None):
    """One batched non-blocking send and/or receive (PAPER.md:117 'non-blocking send and receive'); returns the requests."""
    ops = []
    if send_to is not None:
        ops.append(dist.P2POp(dist.isend, send_tensor, send_to, group))
    if recv_from is not None:
        ops.append(dist.P2POp(dist.irecv, recv_tensor, recv_from, group))
    return dist.batch_isend_irecv(ops) if ops else []


def _wait(reqs):
    for r in reqs:
        r.wait()


class _Staged:
    """A halo exchange that goes through host memory (host_staging): the requests, and the copy of the received host
    tensor into the device tensor that has to follow their completion."""

    def __init__(self, reqs, host, dev):
        self.reqs, self.host, self.dev = reqs, host, dev

    def wait(self):
        _wait(self.reqs)
        if self.dev is not None:
            self.dev.copy_(self.host)


class BlockPath:
    """One rank's share of a sharded evaluation.  rank/world default to the default process group's; world = 1 needs no
    process group at all (the block is the whole path).
    host_staging: device halos travel as host copies (send: device -> host, receive: host -> device) and the 8-byte
    reduction runs on a host tensor, so that a process group without device support (gloo) can drive GPU engines -- the
    functional multi-rank run on ONE GPU (bench.py --dist-backend gloo --all-ranks-on-one-gpu); slower, same results."""

    def __init__(self, engine, n_atoms, first_bead, n_beads, n_beads_path, rank=None, world=None, device="cpu",
                 dtype=torch.float32, group=None, host_staging=False):
        self.host_staging = bool(host_staging)
        self.engine = engine
        self.world = world if world is not None else (dist.get_world_size(group) if dist.is_initialized() else 1)
        self.rank = rank if rank is not None else (dist.get_rank(group) if dist.is_initialized() else 0)
        self.group = group
        self.first, self.n, self.n_path = int(first_bead), int(n_beads), int(n_beads_path)
        self.has_left = self.first > 0
        self.has_right = self.first + self.n < self.n_path
        self.left = self.rank - 1 if self.has_left else None
        self.right = self.rank + 1 if self.has_right else None
        mk = lambda: torch.zeros((n_atoms, 3), dtype=dtype, device=device)
        self.R_right, self.keta_out, self.keta_left = mk(), mk(), mk()
        self._vbuf = torch.zeros(1, dtype=torch.float64, device="cpu" if self.host_staging else device)
        self._h_recv = torch.zeros((n_atoms, 3), dtype=dtype) if self.host_staging else None

    def _halo(self, send_to, send_tensor, recv_from, recv_tensor):
        """Non-blocking exchange of one halo each way; returns something with .wait()."""
        if not self.host_staging:
            return _Staged(_exchange(send_to, send_tensor, recv_from, recv_tensor, self.group), None, None)
        h_send = send_tensor.cpu() if send_to is not None else None     # synchronises this rank's stream: the halo is ready
        reqs = _exchange(send_to, h_send, recv_from, self._h_recv, self.group)
        return _Staged(reqs, self._h_recv, recv_tensor if recv_from is not None else None)

    def eval(self, R_block, grad_out=None, sync=True):
        """R_block [n_beads][Q][3] (this rank's beads).  Returns (V_eff of the WHOLE path, gradient of this block).
        sync=False: the assembly stays asynchronous and no V_eff is formed (returns (None, gradient)): a stepping loop needs
        the gradient only; read the energy when it is wanted with veff()."""
        # 1. right halo of the coordinates
        self._halo(self.left, R_block[0].contiguous(), self.right, self.R_right).wait()
        # 2. pass 1
        self.engine.mop_block_pass1(R_block, self.R_right if self.has_right else None,
                                    self.keta_out if self.has_right else None)
        # 3. K eta halo in flight during pass 2
        halo = self._halo(self.right, self.keta_out, self.left, self.keta_left)
        # 4. pass 2
        self.engine.mop_block_pass2(R_block)
        halo.wait()
        # 5. assembly and the 8-byte reduction
        if not sync:
            return self.engine.mop_block_assemble(self.keta_left if self.has_left else None, grad_out, sync=False)
        v_local, grad = self.engine.mop_block_assemble(self.keta_left if self.has_left else None, grad_out)
        return self._reduce(v_local), grad

    def veff(self):
        """V_eff of the whole path at the last evaluation (synchronises this rank's stream; 8-byte all-reduce)."""
        return self._reduce(self.engine.mop_get_stats()["veff"])

    def _reduce(self, v_local):
        if self.world > 1:
            self._vbuf[0] = v_local
            dist.all_reduce(self._vbuf, op=dist.ReduceOp.SUM, group=self.group)
            v_local = float(self._vbuf.item())
        return v_local
