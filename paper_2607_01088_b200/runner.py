"""Marshalling helpers shared by tests, bench.py and smoke(): put a ``cases.Case`` on the
device and call the C-ABI.  No arithmetic of the method happens here."""
from __future__ import annotations

from typing import List, Optional, Tuple

import numpy as np
import torch

from . import binding as rosa
from .cases import Case


class LoadedCase:
    """An expert created from ``case.weights`` with every robot's prefix K/V bound.

    bf16 cases: per layer ONE packed ragged device buffer [sum L_i, n_kv, hd] bf16, robot i
    bound at offset cu_seqlens[i] (BASELINE.json cfg2 "packed ragged with cu_seqlens offsets").
    fp32 cases (cfg0): per-robot float32 tensors, converted by the library at bind time.
    """

    def __init__(self, case: Case, device: str = "cuda:0", max_batch: Optional[int] = None,
                 max_steps: int = 16):
        self.case = case
        self.device = torch.device(device)
        cfg = case.cfg
        B = case.batch
        max_len = int(case.prefix_lens.max()) if B else 0
        with torch.cuda.device(self.device):
            self.expert = rosa.rosa_expert_create(cfg.as_dict(), case.weights, max_robots=B,
                                                  max_batch=max_batch or B, max_prefix_len=max_len,
                                                  max_steps=max_steps)
            self.kv_buffers: List[torch.Tensor] = []
            cu = case.cu_seqlens()
            row = cfg.n_kv_heads * cfg.head_dim
            if case.bf16:
                kl, vl = [], []
                for l in range(cfg.layers):
                    k = np.concatenate([case.prefix_k[i][l] for i in range(B)], axis=0)
                    v = np.concatenate([case.prefix_v[i][l] for i in range(B)], axis=0)
                    kl.append(torch.from_numpy(k.view(np.int16)).to(self.device).view(torch.bfloat16))
                    vl.append(torch.from_numpy(v.view(np.int16)).to(self.device).view(torch.bfloat16))
                self.kv_buffers = kl + vl
                # per robot: (K pointers per layer, V pointers per layer, length) into the packed buffers
                self.bind_args = [([t.data_ptr() + int(cu[i]) * row * 2 for t in kl],
                                   [t.data_ptr() + int(cu[i]) * row * 2 for t in vl], int(case.prefix_lens[i]))
                                  for i in range(B)]
                self.rebind_all()
            else:
                for i in range(B):
                    ks = [torch.from_numpy(np.ascontiguousarray(case.prefix_k[i][l])).to(self.device)
                          for l in range(cfg.layers)]
                    vs = [torch.from_numpy(np.ascontiguousarray(case.prefix_v[i][l])).to(self.device)
                          for l in range(cfg.layers)]
                    rosa.rosa_prefix_kv_bind(self.expert, i, ks, vs, int(case.prefix_lens[i]), rosa.ROSA_F32)
            torch.cuda.synchronize(self.device)

    def rebind_all(self):
        """rosa_prefix_kv_bind for every robot of a bf16 case (what a serving loop does when each request carries a
        new observation): borrowed pointers, no copy."""
        for i, (kp, vp, length) in enumerate(self.bind_args):
            rosa.rosa_prefix_kv_bind(self.expert, i, kp, vp, length, rosa.ROSA_BF16)

    def kv_bytes(self) -> int:
        return sum(t.numel() * t.element_size() for t in self.kv_buffers)

    def run(self, robots=None, want_velocity: bool = False, stream=None
            ) -> Tuple[np.ndarray, Optional[np.ndarray]]:
        """One rosa_denoise_batch_ex call on the case's own (t_start, dt, n_steps)."""
        c = self.case
        idx = np.arange(c.batch) if robots is None else np.asarray(robots)
        with torch.cuda.device(self.device):
            noise = torch.from_numpy(np.ascontiguousarray(c.noise[idx])).to(self.device)
            out = torch.empty_like(noise)
            nmax = int(c.n_steps[idx].max())
            vel = torch.empty((nmax,) + tuple(noise.shape), dtype=torch.float32, device=self.device) \
                if want_velocity else None
            rosa.rosa_denoise_batch_ex(self.expert, idx.astype(np.int32), noise, c.t_start[idx], c.dt[idx],
                                       c.n_steps[idx], out, vel, stream)
            torch.cuda.synchronize(self.device)
        return out.cpu().numpy(), (vel.cpu().numpy() if vel is not None else None)

    def close(self):
        rosa.rosa_expert_destroy(self.expert)
        self.kv_buffers = []


def rel_l2(got: np.ndarray, want: np.ndarray) -> float:
    """||got - want||_2 / ||want||_2 over the whole tensor (reading R18)."""
    g = np.asarray(got, dtype=np.float64).ravel()
    w = np.asarray(want, dtype=np.float64).ravel()
    return float(np.linalg.norm(g - w) / max(np.linalg.norm(w), 1e-300))


class DeviceFleet:
    """Timing-only workload (bench.py batch sweep): the weights of a seeded ``Case`` drawn
    without prefix data, and per-robot prefix K/V ~ N(0,1) bf16 drawn ON THE DEVICE with a seeded
    torch generator (values do not affect timing; parity tests always use ``LoadedCase``)."""

    def __init__(self, case: Case, prefix_lens, device: str = "cuda:0", max_steps: int = 16, seed: int = 0):
        self.case = case
        self.device = torch.device(device)
        cfg = case.cfg
        lens = np.asarray(prefix_lens, dtype=np.int32)
        self.lens = lens
        B = int(lens.shape[0])
        self.batch = B
        cu = np.zeros(B + 1, dtype=np.int64)
        np.cumsum(lens, out=cu[1:])
        row = cfg.n_kv_heads * cfg.head_dim
        with torch.cuda.device(self.device):
            self.expert = rosa.rosa_expert_create(cfg.as_dict(), case.weights, max_robots=B, max_batch=B,
                                                  max_prefix_len=int(lens.max()), max_steps=max_steps)
            g = torch.Generator(device=self.device)
            g.manual_seed(seed)
            total = int(cu[-1])
            self.k = [torch.randn((total, row), generator=g, device=self.device, dtype=torch.float32)
                      .to(torch.bfloat16) for _ in range(cfg.layers)]
            self.v = [torch.randn((total, row), generator=g, device=self.device, dtype=torch.float32)
                      .to(torch.bfloat16) for _ in range(cfg.layers)]
            for i in range(B):
                off = int(cu[i]) * row * 2
                rosa.rosa_prefix_kv_bind(self.expert, i, [t.data_ptr() + off for t in self.k],
                                         [t.data_ptr() + off for t in self.v], int(lens[i]), rosa.ROSA_BF16)
            self.noise = torch.randn((B, cfg.horizon, cfg.action_dim), generator=g, device=self.device,
                                     dtype=torch.float32)
            torch.cuda.synchronize(self.device)

    def kv_bytes(self) -> int:
        return sum(t.numel() * t.element_size() for t in self.k + self.v)

    def close(self):
        rosa.rosa_expert_destroy(self.expert)
        self.k, self.v = [], []
