"""CPU test of peer.import_pool's restricted unpickler (a forged handle must be refused, not executed)."""
import io
import os
import pickle

import pytest
import torch
from torch.multiprocessing import reductions

from paper_2504_03775_b200 import peer


def test_forged_handle_is_refused_not_executed(tmp_path):
    marker = tmp_path / "pwned"
    evil = pickle.dumps((os.system, (f"touch {marker}",)))
    with pytest.raises(pickle.UnpicklingError):
        peer.import_pool(evil)
    assert not marker.exists()
    # a handle whose callable is allowed to unpickle but is not the IPC rebuild function is refused as well
    with pytest.raises(pickle.UnpicklingError):
        peer.import_pool(pickle.dumps((torch.Size, ([1],))))


def test_genuine_handle_shape_unpickles():
    """The argument tuple torch.multiprocessing.reductions.reduce_tensor produces for a CUDA uint8 buffer
    (types only; no device needed) passes the restricted unpickler unchanged."""
    args = (torch.Tensor, torch.Size([16]), (1,), 0, torch.UntypedStorage, torch.uint8, torch.device("cuda", 0),
            b"h" * 64, 16, 0, False, b"r" * 64, 0, b"e" * 64, True)
    fn, got = peer._HandleUnpickler(io.BytesIO(pickle.dumps((reductions.rebuild_cuda_tensor, args)))).load()
    assert fn is reductions.rebuild_cuda_tensor and got == args
