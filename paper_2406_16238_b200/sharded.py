"""Group drivers for the distributed Hamiltonian ("Distributed Hamiltonian for limited memory",
PAPER.md:308-318, Fig. 6): the Cholesky tensor is split over the gamma index among the G members
of a group, every member owns its own walkers.  These classes only order the afqmc_shard_* phases
of include/afqmc.h, route the caller's auxiliary fields to the member that holds the matching
gamma slice and provide the group barrier; all arithmetic and all walker-sized data movement
(Theta push, V_HS partials stored from the GEMM epilogue into the owner's slot) is in the library.

  LocalGroup  every member lives in this process (one device or several with peer access);
              buffers are exchanged as plain device addresses, barrier = stream synchronise.
  DistGroup   one process per member (torch.distributed); buffers are exchanged as CUDA IPC
              handles; barrier = a one-element all-reduce ordered on the member's stream (NCCL),
              or stream synchronise + host barrier (gloo).
"""
from __future__ import annotations

import numpy as np

from . import afqmc


def gamma_slices(n_chol: int, G: int):
    """Contiguous gamma ranges [(g0, g1)] of even length (TMA needs 16-byte strides), as equal
    as possible; the last member takes the remainder."""
    if n_chol % 2 or G < 1 or n_chol < 2 * G:
        raise ValueError("n_chol must be even and at least 2 per member")
    pairs = n_chol // 2
    base, extra = divmod(pairs, G)
    out, g = [], 0
    for r in range(G):
        n = 2 * (base + (1 if r < extra else 0))
        out.append((g, g + n))
        g += n
    return out


def fields_for_member(x_by_owner, sl):
    """x of every group walker (owner-major) restricted to the gamma slice `sl` = (g0, g1).
    x_by_owner: list of [nw][n_chol_total] arrays/tensors, one per member."""
    import torch
    parts = [torch.as_tensor(x)[:, sl[0]:sl[1]] for x in x_by_owner]
    return torch.cat(parts, dim=0).contiguous()


def exchange_fields(x_own, slices, group=None):
    """One process per member: gather every member's fields and keep the column block of MY gamma
    slice; returns [G * nw][n_local] in owner-major order (the same array `fields_for_member`
    builds when all fields are in one process).  The fields are small (nw * n_chol doubles per
    member), so an all-gather serves; gloo exchanges host tensors, NCCL device tensors."""
    import torch
    import torch.distributed as dist
    rank = dist.get_rank(group)
    if dist.get_backend(group) == "gloo" and x_own.is_cuda:
        raise ValueError("gloo exchanges host tensors: pass the fields as a CPU tensor")
    x_own = x_own.contiguous()
    everyone = [torch.empty_like(x_own) for _ in slices]
    dist.all_gather(everyone, x_own, group=group)
    return fields_for_member(everyone, slices[rank])


class LocalGroup:
    """G members in one process.  L_slices[r] is member r's device tensor [n_r][M][M]."""

    def __init__(self, h1, L_slices, trial, *, M, n_alpha, n_beta, max_walkers, walker_kind,
                 taylor_order=6, ortho_every=0, e_shift=None, pack_chol=False):
        self.G = len(L_slices)
        self.nw = max_walkers
        self.slices, g = [], 0
        for Ls in L_slices:
            self.slices.append((g, g + int(Ls.shape[0])))
            g += int(Ls.shape[0])
        self.n_chol = g
        self.members = [
            afqmc.AFQMC(h1, Ls, trial, M=M, n_alpha=n_alpha, n_beta=n_beta, n_chol=int(Ls.shape[0]),
                        max_walkers=max_walkers, walker_kind=walker_kind, taylor_order=taylor_order,
                        ortho_every=ortho_every, e_shift=e_shift, pack_chol=pack_chol,
                        group_size=self.G, group_rank=r)
            for r, Ls in enumerate(L_slices)]
        # setup sums in member order 0..G-1 (added up inside the library), the same on every member
        total = afqmc.AFQMC.shard_setup_reduce(np.stack([m.shard_setup_partial() for m in self.members]))
        addrs = np.stack([m.shard_get_buffers() for m in self.members])
        for m in self.members:
            m.shard_setup_finish(total)
            m.shard_set_peers(addrs)

    def barrier(self):
        for m in self.members:
            m.sync()

    def step(self, walkers, weights, x_by_owner, dt):
        """walkers[r] [nw][M][Nt] c128, weights[r] [nw], x_by_owner[r] [nw][n_chol] (device tensors)."""
        xs = [fields_for_member(x_by_owner, sl) for sl in self.slices]
        self._sync_torch()
        for m, W in zip(self.members, walkers):
            m.shard_theta(W, for_energy=False)
        self.barrier()
        for m, x in zip(self.members, xs):
            m.shard_vhs(x, dt, self.nw)
        self.barrier()
        for m, W, wt in zip(self.members, walkers, weights):
            m.shard_propagate(W, wt, dt)
        self.barrier()

    def local_energy(self, walkers, E_out):
        self._sync_torch()
        for m, W in zip(self.members, walkers):
            m.shard_theta(W, for_energy=True)
        self.barrier()
        for m in self.members:
            m.shard_energy(self.nw)
        self.barrier()
        for m, E in zip(self.members, E_out):
            m.shard_energy_finish(E)
        self.barrier()

    @staticmethod
    def _sync_torch():
        import torch
        torch.cuda.synchronize()     # the members run on their own streams, torch on another

    def close(self):
        for m in self.members:
            m.close()
        self.members = []


class DistGroup:
    """One process per member.  `L_local` is this member's slice [n_local][M][M] on its device;
    `slices` the gamma ranges of all members (gamma_slices)."""

    def __init__(self, h1, L_local, trial, slices, *, M, n_alpha, n_beta, max_walkers, walker_kind,
                 taylor_order=6, ortho_every=0, e_shift=None, pack_chol=False, group=None):
        import torch
        import torch.distributed as dist
        self.dist, self.torch, self.group = dist, torch, group
        self.G, self.rank = dist.get_world_size(group), dist.get_rank(group)
        self.slices, self.nw = list(slices), max_walkers
        assert len(self.slices) == self.G and self.slices[self.rank][1] - self.slices[self.rank][0] == L_local.shape[0]
        self.nccl = dist.get_backend(group) == "nccl"
        self.stream = torch.cuda.Stream()
        self.member = afqmc.AFQMC(h1, L_local, trial, M=M, n_alpha=n_alpha, n_beta=n_beta,
                                  n_chol=int(L_local.shape[0]), max_walkers=max_walkers, walker_kind=walker_kind,
                                  taylor_order=taylor_order, ortho_every=ortho_every, e_shift=e_shift,
                                  pack_chol=pack_chol, stream=self.stream.cuda_stream,
                                  group_size=self.G, group_rank=self.rank)
        # setup sums: all-reduce (every member gets the same bits)
        part = torch.from_numpy(self.member.shard_setup_partial())
        if self.nccl:
            part = part.cuda()
        dist.all_reduce(part, group=group)
        self.member.shard_setup_finish(part.cpu().numpy())
        # peer buffers through CUDA IPC
        mine = [self.member.shard_ipc_export(k).tobytes() for k in range(4)]
        everyone = [None] * self.G
        dist.all_gather_object(everyone, mine, group=group)
        own = self.member.shard_get_buffers()
        addrs = np.zeros((self.G, 4), dtype=np.uint64)
        self._opened = []
        for r in range(self.G):
            for k in range(4):
                if r == self.rank:
                    addrs[r, k] = own[k]
                else:
                    addrs[r, k] = self.member.shard_ipc_open(everyone[r][k])
                    self._opened.append(int(addrs[r, k]))
        self.member.shard_set_peers(addrs)
        self._flag = torch.zeros(1, device="cuda") if self.nccl else None
        self.barrier()

    def barrier(self):
        if self.nccl:      # ordered on the member's stream, no host synchronisation
            with self.torch.cuda.stream(self.stream):
                self.dist.all_reduce(self._flag, group=self.group)
        else:
            self.member.sync()
            self.dist.barrier(group=self.group)

    def _fields(self, x_own):
        if self.nccl:
            with self.torch.cuda.stream(self.stream):
                return exchange_fields(x_own, self.slices, self.group)
        return exchange_fields(x_own.cpu(), self.slices, self.group).cuda()

    def step(self, walkers, weights, x_own, dt):
        """x_own: this member's fields [nw][n_chol_total] (device tensor)."""
        self.torch.cuda.current_stream().synchronize()
        x = self._fields(x_own)
        if not self.nccl:
            self.torch.cuda.synchronize()
        self.member.shard_theta(walkers, for_energy=False)
        self.barrier()
        self.member.shard_vhs(x, dt, self.nw)
        self.barrier()
        self.member.shard_propagate(walkers, weights, dt)
        self._keep = x                 # alive until the stream has consumed it

    def local_energy(self, walkers, E_out):
        self.torch.cuda.current_stream().synchronize()
        self.member.shard_theta(walkers, for_energy=True)
        self.barrier()
        self.member.shard_energy(self.nw)
        self.barrier()
        self.member.shard_energy_finish(E_out)

    def sync(self):
        self.member.sync()

    def close(self):
        if self.member is not None:
            self.member.sync()
            self.dist.barrier(group=self.group)      # nobody may still be writing into my slots
            for a in self._opened:
                afqmc.lib.afqmc_shard_ipc_close(a)
            self.member.close()
            self.member = None
