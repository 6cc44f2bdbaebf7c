"""Device-memory plumbing for the binding: PyTorch owns the buffers and the stream, libaceapex does the work."""
from __future__ import annotations

import numpy as np
import torch

from . import PHASE_ALL, Plan


class Decoder:
    """One compressed buffer resident on the GPU + output and scratch tensors; ``run`` enqueues aceapex_decode."""

    def __init__(self, comp: np.ndarray, device: int = 0, strategy: int = 0):
        assert comp.dtype == np.uint8 and comp.flags.c_contiguous
        if not torch.cuda.is_available():
            raise RuntimeError("aceapex needs a CUDA device (no CPU fallback)")
        self.comp_host = comp
        self.plan = Plan(comp.ctypes.data, comp.size, device)
        if strategy:
            self.plan.set_strategy(strategy)
        self.dev = torch.device("cuda", device)
        self.comp_dev = torch.from_numpy(comp).to(self.dev) if comp.size else torch.empty(0, dtype=torch.uint8, device=self.dev)
        self.out_dev = torch.zeros(max(self.plan.out_bytes, 16), dtype=torch.uint8, device=self.dev)
        self.scratch = torch.empty(max(self.plan.scratch_bytes, 16), dtype=torch.uint8, device=self.dev)

    def run(self, phases: int = PHASE_ALL):
        st = torch.cuda.current_stream(self.dev).cuda_stream
        self.plan.decode(self.comp_dev.data_ptr(), self.out_dev.data_ptr(), self.out_dev.numel(), self.scratch.data_ptr(),
                         self.scratch.numel(), phases, st)

    def output(self) -> np.ndarray:
        torch.cuda.synchronize(self.dev)
        return self.out_dev[: self.plan.raw_bytes].cpu().numpy()

    def stats(self, check: bool = True) -> dict:
        return self.plan.stats(self.scratch.data_ptr(), check=check)

    def close(self):
        self.plan.close()


def decode(comp: np.ndarray, device: int = 0, strategy: int = 0) -> np.ndarray:
    """Decode one stream and return the bytes (raises AceapexError on any fault, including device-side ones)."""
    d = Decoder(comp, device, strategy)
    try:
        d.run()
        out = d.output()
        d.stats(check=True)
        return out
    finally:
        d.close()
