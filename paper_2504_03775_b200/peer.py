"""Peer pools over CUDA IPC — the paper's single-machine "IPC" mode.

A decode-side process owns its KV pool and exports it; the prefill-side process maps it and runs the SAME
``flowkv_transfer`` kernel with the mapped pointer as the dst pool: a one-sided put, no collective, no
staging buffer, no receiver-side kernel.  On a multi-GPU node the mapping crosses NVLink; with one GPU both
processes share the device and the stores land in the same HBM.

torch is used for what it is here for — device memory and its IPC plumbing (``cudaIpcGetMemHandle`` /
``cudaIpcOpenMemHandle`` behind ``torch.multiprocessing.reductions``); no KV byte is moved by torch.
"""
from __future__ import annotations

import pickle

import torch
from torch.multiprocessing import reductions


def export_pool(buf: torch.Tensor) -> bytes:
    """Serialise an IPC handle of a CUDA uint8 buffer.  The exporting process must keep ``buf`` alive (and stay
    alive itself) for as long as any importer uses the mapping."""
    assert buf.is_cuda and buf.dtype == torch.uint8 and buf.is_contiguous()
    fn, args = reductions.reduce_tensor(buf)
    return pickle.dumps((fn, args))


class _HandleUnpickler(pickle.Unpickler):
    """Unpickles an export_pool() handle and nothing else: the only globals a handle may name are torch's CUDA-IPC
    rebuild function, torch.device / dtype objects and the storage classes its argument tuple carries.  Anything
    else (``os.system``, ``builtins.eval`` ...) is refused instead of being called."""
    _ALLOWED = {("torch.multiprocessing.reductions", "rebuild_cuda_tensor"), ("torch", "device"), ("torch", "Size"),
                ("torch", "uint8"), ("torch", "Tensor"), ("torch", "UntypedStorage"), ("torch.storage", "UntypedStorage"),
                ("torch", "TypedStorage"), ("torch.storage", "TypedStorage")}

    def find_class(self, module, name):
        if (module, name) not in self._ALLOWED:
            raise pickle.UnpicklingError(f"peer handle names {module}.{name}: not a CUDA-IPC pool handle")
        return super().find_class(module, name)


def import_pool(handle: bytes) -> torch.Tensor:
    """Map an exported buffer into this process; ``.data_ptr()`` is what ``flowkv.make_pool`` takes.
    The mapping lives as long as the returned tensor.

    ``handle`` must come from :func:`export_pool` in another process ON THE SAME MACHINE.  It is unpickled with a
    restricted unpickler (only torch's CUDA-IPC rebuild function and its plain arguments are accepted), so a forged
    handle is rejected rather than executed; mapping another process's memory still requires trusting that process
    with the bytes this GPU writes there."""
    import io
    fn, args = _HandleUnpickler(io.BytesIO(handle)).load()
    if fn is not reductions.rebuild_cuda_tensor:
        raise pickle.UnpicklingError("peer handle does not rebuild a CUDA tensor")
    t = fn(*args)
    assert t.is_cuda and t.dtype == torch.uint8
    return t
