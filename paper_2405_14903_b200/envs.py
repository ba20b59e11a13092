"""Many small environments at once (the paper's tasks are 40^3-48^3 grids, far
too small to fill a B200 one at a time): one nf_grid handle + CUDA stream + host thread per environment.  A solve's
host side only launches kernels and polls a mapped status word, and ctypes releases the GIL around every C-ABI call, so
E threads keep E streams busy; on the device the kernels of different environments overlap (the cooperative coarse
kernel is sized for its level, not for the machine: csrc/nf_mg.cu nf_mg_init).  Plumbing only -- no arithmetic."""
import threading

import torch

from . import api


class EnvPool:
    """E independent grids of the same shape.  run(fn) calls fn(index, grid) for every environment concurrently, each
    on its own stream (made current for torch ops inside fn), and returns the list of results."""

    def __init__(self, n_envs, nx, ny, nz, dx, device=None):
        self.grids = [api.Grid(nx, ny, nz, dx, device) for _ in range(int(n_envs))]
        self.device = self.grids[0].device
        self.streams = [torch.cuda.Stream(device=self.device) for _ in self.grids]
        for g, s in zip(self.grids, self.streams):
            g.set_stream(s)

    def __len__(self):
        return len(self.grids)

    def run(self, fn):
        out = [None] * len(self.grids)
        err = [None] * len(self.grids)

        def work(i):
            try:
                with torch.cuda.device(self.device), torch.cuda.stream(self.streams[i]):
                    out[i] = fn(i, self.grids[i])
            except BaseException as e:  # re-raised in the caller's thread
                err[i] = e

        threads = [threading.Thread(target=work, args=(i,)) for i in range(len(self.grids))]
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        for e in err:
            if e is not None:
                raise e
        return out

    def synchronize(self):
        for s in self.streams:
            s.synchronize()

    def close(self):
        self.synchronize()
        for g in self.grids:
            g.close()
        self.grids = []
