"""Halo exchange of the decomposed sweep (reading P-21 in DESIGN.md): plumbing only.

One process per GPU holds the LOCAL grid of its rank (``IconGrid(k, n_parts=R, part=r)``). Before a step the halo rows
of ``vn`` and ``w`` are filled from their owners:

    pack      dycore_halo_pack (the library's kernel): the owned rows the peers read, gathered into ONE contiguous
              buffer laid out [rows for rank 0 | rows for rank 1 | ...]
    transport ONE ``all_to_all_single`` per field over the process group (NCCL: grouped send / recv over NVLink;
              the point-to-point exchange of PAPER.md:97-105), split sizes from the grid's tables
    receive   straight into the halo rows of the local field, which the local numbering makes one contiguous block
              per peer in rank order: nothing is unpacked

There is no arithmetic here. Everything a step computes runs in the library's kernels on the local grid.
"""
import numpy as np

from . import binding


class HaloExchange:
    """Split sizes and buffers of one rank's exchange. ``group`` is a torch.distributed process group whose rank r
    holds part r (None = the default group)."""

    def __init__(self, grid, group=None):
        info = grid.part_info()
        if not info["n_parts"]:
            raise ValueError("HaloExchange needs a grid made with n_parts > 0")
        self.grid, self.group, self.info = grid, group, info
        self.n_owned = (info["ne_owned"], info["nc_owned"])
        self.n_local = (info["ne_local"], info["nc_local"])
        self.recv_rows, self.send_rows = [], []
        for kind, name in enumerate(("edge", "cell")):
            rb = grid.part_table("recv_begin_" + name)
            sb = grid.part_table("send_begin_" + name)
            self.recv_rows.append([int(x) for x in np.diff(rb)])
            self.send_rows.append([int(x) for x in np.diff(sb)])
            assert int(rb[0]) == self.n_owned[kind] and int(rb[-1]) == self.n_local[kind]
        self._buf = {}

    def send_buffer(self, kind, like):
        """[n_send][ld] buffer with the dtype, device and row stride of the field `like` (cached per shape)"""
        n = sum(self.send_rows[kind])
        key = (kind, like.dtype, like.device, like.shape[1])
        b = self._buf.get(key)
        if b is None:
            b = like.new_empty((n, like.shape[1]))
            self._buf[key] = b
        return b

    def exchange(self, field, kind, pack=None, async_op=False):
        """fills rows [n_owned, n_local) of `field` ([n_local][ld], contiguous) with their owners' rows. kind 0 = edge
        field (vn), 1 = cell field (w). `pack(grid, kind, field, send_buf)` defaults to the library's kernel on the
        current CUDA stream (the CPU tests of the plumbing pass a host gather). Returns the work handle if async_op."""
        import torch.distributed as dist
        if field.shape[0] != self.n_local[kind] or not field.is_contiguous():
            raise ValueError("field must be a contiguous [n_local][ld] tensor of the local grid")
        if dist.get_world_size(self.group) != self.info["n_parts"] or dist.get_rank(self.group) != self.info["part"]:
            raise ValueError("the process group does not match the grid's (n_parts, part)")
        ld = field.shape[1]
        send = self.send_buffer(kind, field)
        (pack or binding.dycore_halo_pack)(self.grid, kind, field, send)
        halo = field[self.n_owned[kind]:]
        return dist.all_to_all_single(halo.reshape(-1), send.reshape(-1),
                                      output_split_sizes=[r * ld for r in self.recv_rows[kind]],
                                      input_split_sizes=[r * ld for r in self.send_rows[kind]],
                                      group=self.group, async_op=async_op)
