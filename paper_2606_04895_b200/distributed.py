"""torch.distributed plumbing for the one exchange step of the sharded path (include/best.h
best_set_adaptation_exchange): at the end of every covariance window each rank's packet of window sums is
all-gathered, rank order, and the library combines them on the device.  No arithmetic of the method here: the
functions only move the library's packets through NCCL (gloo in the CPU tests)."""
import torch
import torch.distributed as dist


def allgather_packets(send: torch.Tensor, recv: torch.Tensor, group=None) -> None:
    """recv[r * n : (r + 1) * n] = rank r's `send` (n = send.numel()); device tensors over NCCL, CPU tensors over gloo."""
    assert recv.numel() == send.numel() * dist.get_world_size(group)
    if send.is_cuda:
        dist.all_gather_into_tensor(recv, send, group=group)
    else:   # gloo has no all_gather_into_tensor for flat outputs on every version: gather into views
        dist.all_gather(list(recv.view(dist.get_world_size(group), -1).unbind(0)), send, group=group)


class _DevMem:
    """Zero-copy view of library-owned device memory for torch.as_tensor (CUDA array interface)."""

    def __init__(self, ptr: int, count: int):
        self.__cuda_array_interface__ = {"shape": (count,), "typestr": "<f8", "data": (ptr, False), "version": 3}


def device_view(ptr: int, count: int) -> torch.Tensor:
    return torch.as_tensor(_DevMem(ptr, count), device="cuda")


def allgather_exchange(group=None):
    """The callable State.set_adaptation_exchange expects: all-gathers the packets on the library's stream."""
    world = dist.get_world_size(group)

    def fn(send_ptr, recv_ptr, count, stream):
        send, recv = device_view(send_ptr, count), device_view(recv_ptr, count * world)
        with torch.cuda.stream(torch.cuda.ExternalStream(stream) if stream else torch.cuda.default_stream()):
            allgather_packets(send, recv, group)
        return 0
    return fn
