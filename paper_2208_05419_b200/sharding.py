"""Multi-GPU use of the AFNO spectral layer: host-side index logic only.

The layer shards two ways (Fig. 2 caption :119), neither of which puts a collective INSIDE it:

* by sample (data parallelism): every rank runs the layer on its own samples; "weight gradients need to be reduced
  across all model instances": dW1, db1, dW2, db2 are SUMS over the samples, so one all-reduce(SUM)
  of 1.19 MB at 768 channels.  `GradBucket` keeps the four gradient tensors as views of ONE flat fp32 buffer, so
  the step issues a single NCCL all-reduce on the layer's stream right behind `afno_spectral_bwd`.
* by channel block (the paper's feature parallelism): "we can distribute the blocks across the GPUs ... embarrassingly
  parallel": rank r owns blocks [j0, j0 + n) = channels [j0 bs, (j0 + n) bs) of x, y, dY, dX and the
  matching slices of the parameters; no collective at all.

Everything numeric runs in the kernels of libafno_b200.so through `binding`; this module holds no arithmetic of the
method.  One process per GPU (`torch.distributed`, NCCL over NVLink); the functions take the process group as an
argument so that the CPU tests can drive the same logic with gloo.
"""
from __future__ import annotations

from dataclasses import dataclass


def split_range(n: int, rank: int, world: int):
    """Contiguous, balanced split of range(n) over `world` ranks: (start, count) of `rank` (the first n % world
    ranks get one more)."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("rank / world out of range")
    base, extra = divmod(n, world)
    start = rank * base + min(rank, extra)
    return start, base + (1 if rank < extra else 0)


def shard_batch(B: int, rank: int, world: int):
    """Data parallelism: samples [b0, b0 + n) of a global batch of B."""
    return split_range(B, rank, world)


def shard_blocks(num_blocks: int, C: int, rank: int, world: int):
    """Feature parallelism: blocks [j0, j0 + n) and the channel range [c0, c0 + nc) they cover."""
    if C % num_blocks:
        raise ValueError("num_blocks must divide C")
    bs = C // num_blocks
    j0, n = split_range(num_blocks, rank, world)
    return j0, n, j0 * bs, n * bs


def param_shapes(num_blocks: int, bs: int, hidden_factor: int = 1):
    """Shapes of (w1, b1, w2, b2) = of (dw1, db1, dw2, db2), reading A11: [nb, in, out, 2] / [nb, out, 2]."""
    hid = bs * hidden_factor
    return [(num_blocks, bs, hid, 2), (num_blocks, hid, 2), (num_blocks, hid, bs, 2), (num_blocks, bs, 2)]


@dataclass
class GradBucket:
    """dw1, db1, dw2, db2 as views of one flat fp32 tensor (offsets rounded up to 16 bytes, the C ABI's alignment)."""
    flat: object
    views: list

    @staticmethod
    def offsets(shapes):
        offs, off = [], 0
        for s in shapes:
            n = 1
            for d in s:
                n *= d
            offs.append((off, n))
            off = (off + n + 3) // 4 * 4      # 4 floats = 16 bytes
        return offs, off

    @classmethod
    def allocate(cls, num_blocks: int, bs: int, hidden_factor: int = 1, device="cuda"):
        import torch
        shapes = param_shapes(num_blocks, bs, hidden_factor)
        offs, total = cls.offsets(shapes)
        flat = torch.zeros(total, dtype=torch.float32, device=device)
        return cls(flat, [flat[o:o + n].view(s) for (o, n), s in zip(offs, shapes)])

    def all_reduce(self, dist, group=None, stream=None):
        """Sum over the data-parallel ranks: NCCL enqueues it, gloo blocks.

        `stream`: the stream the gradients were written on (torch.cuda.Stream or a raw handle).  torch.distributed orders
        an NCCL collective only against torch's CURRENT stream, so the collective is issued with `stream` made current:
        it then runs behind the backward kernels that fill the bucket, whichever stream the caller has current.  None =
        the caller's current stream (right only when the backward was enqueued there)."""
        if dist is not None and dist.get_world_size(group) > 1:
            if stream is not None and getattr(self.flat, "is_cuda", False):
                import torch
                s = torch.cuda.ExternalStream(stream) if isinstance(stream, int) else stream
                with torch.cuda.stream(s):
                    dist.all_reduce(self.flat, op=dist.ReduceOp.SUM, group=group)
            else:
                dist.all_reduce(self.flat, op=dist.ReduceOp.SUM, group=group)
        return self.views


def slice_params_for_blocks(params, j0: int, n: int):
    """Parameter (or gradient) tensors of blocks [j0, j0 + n): the leading axis is the block (reading A11)."""
    return [p[j0:j0 + n] for p in params]


def data_parallel_step(binding, desc_local, x, dy, params, y, dx, bucket: GradBucket, ws, stream, dist=None, group=None):
    """One training step of the layer on this rank's samples, then ONE all-reduce of the parameter gradients.

    desc_local: descriptor with B = this rank's sample count.  The forward saves its context in `ws`, the backward
    reads it (S1).  `stream` (None = the current stream) carries all three: forward, backward and the
    collective.  Returns the launch count of the two calls."""
    d_f = binding.Desc(**{**desc_local.__dict__, "flags": desc_local.flags | binding.FLAG_SAVE_CONTEXT})
    d_b = binding.Desc(**{**desc_local.__dict__, "flags": desc_local.flags | binding.FLAG_USE_CONTEXT})
    binding.afno_spectral_fwd(d_f, x, *params, y, ws, stream)
    n = binding.afno_last_launch_count()
    binding.afno_spectral_bwd(d_b, x, dy, *params, dx, *bucket.views, ws, stream)
    n += binding.afno_last_launch_count()
    bucket.all_reduce(dist, group, stream)     # on `stream`, behind the backward, not on whatever stream is current
    return n
