"""The LP chain over real GPUs, one process per GPU (``lp_chain_*`` of include/lp_collectives.h).

``ChainGroup`` is the multi-process plumbing around one rank's endpoint: every rank creates its endpoint on its own
device, the CUDA IPC handles are all-gathered over ``torch.distributed`` (any backend: the handles are 64 opaque bytes),
every rank maps the endpoints of ranks (rank +- 1) mod P, and from then on a collective is one kernel launch per rank
that pushes blocks into the neighbours' rings over NVLink -- no NCCL call on the data path.  Argument marshalling only:
the chain itself runs in csrc/lp_chain.cu.

This build's box has one GPU, so what runs on it is ``binding.lp_chain_emulate`` (all P ranks in one cooperative
launch); here, the handle exchange and the roles are covered by world_size-2 gloo tests on the CPU
(tests/test_dist_host.py) with a stand-in endpoint, which is why the endpoint factory is a parameter.
"""
from __future__ import annotations

from . import binding as lp


def exchange_handles(my_handle: bytes, group=None):
    """All-gather of one opaque handle per rank, returned in rank order (works on gloo and nccl alike)."""
    import torch.distributed as dist
    world = dist.get_world_size(group)
    out = [None] * world
    dist.all_gather_object(out, bytes(my_handle), group=group)
    if any(h is None or len(h) != len(my_handle) for h in out):
        raise RuntimeError("handle exchange: a rank sent a handle of another size")
    return out


class ChainGroup:
    """One rank's view of the chain: ``ChainGroup()`` after ``torch.distributed`` is initialised and the rank's CUDA
    device is current; then ``allreduce(buf)``, ``reduce(buf, root)``, ``broadcast(buf, root)`` on float32 CUDA tensors
    of the same length on every rank, in the same order on every rank (they are collectives)."""

    def __init__(self, group=None, channels=0, slots=0, tile=0, endpoint_factory=None):
        import torch.distributed as dist
        self.group = group
        self.rank = dist.get_rank(group)
        self.world = dist.get_world_size(group)
        make = endpoint_factory or lp.Chain
        self.endpoint = make(self.rank, self.world, channels, slots, tile)
        self.handles = exchange_handles(self.endpoint.handle(), group)
        self.endpoint.connect(self.handles)
        dist.barrier(group)  # nobody pushes into an endpoint that is not mapped everywhere yet

    def role(self, op, root=0) -> dict:
        return lp.lp_chain_plan(op, self.world, root, self.rank)

    def allreduce(self, buf, block=0, reduce_op=lp.REDUCE_SUM, stream=None):
        self.endpoint.run(lp.OP_ALLREDUCE, buf, block=block, root=0, reduce_op=reduce_op, stream=stream)

    def reduce(self, buf, root=0, block=0, reduce_op=lp.REDUCE_SUM, stream=None):
        self.endpoint.run(lp.OP_REDUCE, buf, block=block, root=root, reduce_op=reduce_op, stream=stream)

    def broadcast(self, buf, root=0, block=0, stream=None):
        self.endpoint.run(lp.OP_BROADCAST, buf, block=block, root=root, stream=stream)

    def bsp_sgd_step(self, grad, weight, lr, block=0, stream=None):
        """Alg. 3: allreduce of the sub-gradients, w -= lr * mean gradient, fused; every rank's `weight` gets the new bits."""
        self.endpoint.bsp_sgd_step(grad, weight, block=block, lr=lr, stream=stream)

    def bsp_sgd_momentum_step(self, grad, weight, velocity, lr, mu, block=0, stream=None):
        """The same with momentum (the paper's solver); `velocity` is the LAST rank's vector, None elsewhere."""
        self.endpoint.bsp_sgd_momentum_step(grad, weight, velocity, block=block, lr=lr, mu=mu, stream=stream)

    def error(self) -> int:
        return self.endpoint.error()

    def destroy(self):
        """Tear-down in the order lp_collectives.h prescribes.  A host barrier alone is not enough: it does not wait for the
        neighbours' KERNELS, and a chain kernel ends without waiting for its last credits -- a neighbour's kernel may
        still be about to store into this rank's endpoint when this rank passes the barrier."""
        import torch
        import torch.distributed as dist
        if torch.cuda.is_available():
            torch.cuda.synchronize()      # 1. my kernels have drained: I push nothing into anybody any more ...
        dist.barrier(self.group)          #    ... and neither does anyone else
        disconnect = getattr(self.endpoint, "disconnect", None)
        if disconnect is not None:
            disconnect()                  # 2. my mappings of the neighbours' endpoints are closed ...
        dist.barrier(self.group)          #    ... and so is every mapping of mine
        self.endpoint.destroy()           # 3. free my (unmapped, idle) endpoint
