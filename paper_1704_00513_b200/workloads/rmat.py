"""R-MAT graphs and BFS frontiers (BASELINE.json configs 1, 3, 4).

Scaffolding only: the thesis's Graph500 generator / GPU BFS (PAPER.md L540, L559-571,
L733-776) are prior work and out of scope; this module just produces the per-level
frontiers (sorted unique vertex IDs) that the codec is fed with. Plain torch integer ops,
device-agnostic (scale 12 on CPU for tests, scale 22/25 on the GPU box), seeded by
workloads/rng.py. No codec arithmetic here.
"""
from __future__ import annotations

import torch

from . import rng

_S_EDGE, _S_ROOT = 0x100, 0x90
# A/B/C/D = .57/.19/.19/.05 as integer thresholds on a 32-bit draw
_T_A = int(0.57 * (1 << 32))
_T_AB = int(0.76 * (1 << 32))
_T_ABC = int(0.95 * (1 << 32))


def rmat_edges(scale: int, n_draws: int, seed: int, device="cpu", chunk: int = 1 << 26):
    """n_draws directed (u, v) pairs, one 32-bit draw per level. Returns int64 keys u*N+v."""
    N = 1 << scale
    keys = []
    for lo in range(0, n_draws, chunk):
        e = torch.arange(lo, min(lo + chunk, n_draws), dtype=torch.int64, device=device)
        u = torch.zeros_like(e)
        v = torch.zeros_like(e)
        for level in range(scale):
            r = rng.u32(seed, _S_EDGE + level, e)
            row = ((r >= _T_AB)).to(torch.int64)                       # C or D quadrant
            col = (((r >= _T_A) & (r < _T_AB)) | (r >= _T_ABC)).to(torch.int64)   # B or D
            u = u * 2 + row
            v = v * 2 + col
        keep = u != v                                                   # drop self-loops
        u, v = u[keep], v[keep]
        keys.append(torch.cat([u * N + v, v * N + u]))                  # symmetrise
        del e, u, v, keep
    return keys


class Graph:
    """CSR of the undirected, deduplicated graph."""

    def __init__(self, scale: int, edgefactor: int, seed: int, device="cpu"):
        self.N = 1 << scale
        self.device = device
        parts = rmat_edges(scale, edgefactor * self.N, seed, device)
        parts = [torch.unique(p) for p in parts]                        # sorted + dedupe per chunk
        keys = torch.unique(torch.cat(parts)) if len(parts) > 1 else parts[0]
        del parts
        src = keys // self.N
        self.col = (keys % self.N).to(torch.int32 if scale < 31 else torch.int64)
        del keys
        deg = torch.bincount(src, minlength=self.N)
        del src
        self.rowptr = torch.zeros(self.N + 1, dtype=torch.int64, device=device)
        self.rowptr[1:] = torch.cumsum(deg, 0)
        self.deg = deg

    def roots(self, n_roots: int, seed: int):
        """candidates rng(seed, t) mod N, keep the first n_roots distinct ones with degree > 0"""
        out, t = [], 0
        deg = self.deg
        while len(out) < n_roots:
            cand = rng.below(seed, _S_ROOT, torch.arange(t, t + 64, dtype=torch.int64), self.N).tolist()
            for c in cand:
                if len(out) < n_roots and c not in out and int(deg[c].item()) > 0:
                    out.append(c)
            t += 64
        return out

    def bfs_frontiers(self, root: int, edge_chunk: int = 1 << 28):
        """level-synchronous BFS; yields each level's newly discovered set as a sorted unique
        int64 tensor (level 0 = [root])."""
        dev = self.device
        visited = torch.zeros(self.N, dtype=torch.bool, device=dev)
        frontier = torch.tensor([root], dtype=torch.int64, device=dev)
        visited[frontier] = True
        while frontier.numel() > 0:
            yield frontier
            start = self.rowptr[frontier]
            deg = self.rowptr[frontier + 1] - start
            found = []
            # expand in chunks of frontier vertices so temporaries stay bounded
            cdeg = torch.cumsum(deg, 0)
            total = int(cdeg[-1].item())
            lo_v = 0
            while lo_v < frontier.numel():
                base = int(cdeg[lo_v - 1].item()) if lo_v else 0
                hi_v = int(torch.searchsorted(cdeg, torch.tensor(base + edge_chunk, device=dev), right=True).item())
                hi_v = max(hi_v, lo_v + 1)
                d = deg[lo_v:hi_v]
                n_e = int(d.sum().item())
                if n_e:
                    excl = torch.cumsum(d, 0) - d
                    idx = (torch.arange(n_e, dtype=torch.int64, device=dev)
                           + torch.repeat_interleave(start[lo_v:hi_v] - excl, d))
                    nb = self.col[idx].to(torch.int64)
                    nb = nb[~visited[nb]]
                    if nb.numel():
                        nb = torch.unique(nb)
                        visited[nb] = True
                        found.append(nb)
                lo_v = hi_v
            del total
            if not found:
                return
            frontier = torch.unique(torch.cat(found)) if len(found) > 1 else found[0]
