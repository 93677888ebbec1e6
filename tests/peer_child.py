"""Decode-side process of the IPC peer-pool test: owns the dst pool, exports it, and reports its bytes after
the prefill-side process has written into it."""
import sys


def decode_side(nbytes: int, sentinel: int, to_parent, from_parent) -> None:
    try:
        import torch
        from paper_2504_03775_b200 import peer
        torch.cuda.set_device(0)
        dst = torch.full((nbytes,), sentinel, dtype=torch.uint8, device="cuda:0")
        torch.cuda.synchronize()
        to_parent.put(("handle", peer.export_pool(dst)))
        msg = from_parent.get(timeout=120)          # the writer has synchronised its stream
        assert msg == "written", msg
        torch.cuda.synchronize()
        to_parent.put(("bytes", dst.cpu().numpy().tobytes()))
        from_parent.get(timeout=120)                # keep the pool alive until the importer has unmapped it
    except Exception as e:  # pragma: no cover
        to_parent.put(("error", repr(e)))
        sys.exit(1)
