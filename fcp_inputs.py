"""Seeded synthetic inputs shared by tests, bench.py and smoke().

This module holds NONE of the method's arithmetic (no planner, no attention, no masks): only
the document-length recipes and the N(0,1) tensors of DESIGN.md section 4 ("input recipe").
They stand in for the paper's WLB-LLM / Pile / RedPajama samples, which are
not available; shapes follow PAPER.md:228 (128K context, head dim 128, 16/32 heads, CP 4/8)
extended by BASELINE.json:configs.  Neither oracle/ nor the CUDA package imports it.
"""

from typing import List, NamedTuple

import numpy as np


class Config(NamedTuple):
    name: str
    C: int          # packed context length
    N: int          # CP size (virtual ranks)
    Hq: int
    Hkv: int
    D: int


CONFIGS = {
    "tiny":     Config("tiny", 1024, 2, 1, 1, 64),
    "8b":       Config("8b", 32768, 4, 32, 8, 128),
    "longtail": Config("longtail", 131072, 8, 32, 8, 128),
    "short":    Config("short", 65536, 16, 32, 8, 128),
    "70b":      Config("70b", 262144, 8, 64, 8, 128),
    # context-window sweep on the long-tail recipe (the shape of the paper's Fig. 7)
    "longtail_64k":  Config("longtail_64k", 65536, 8, 32, 8, 128),
    "longtail_256k": Config("longtail_256k", 262144, 8, 32, 8, 128),
    "longtail_512k": Config("longtail_512k", 524288, 8, 32, 8, 128),
    "longtail_1m":   Config("longtail_1m", 1048576, 8, 32, 8, 128),
    "fig3a":    Config("fig3a", 131072, 8, 32, 8, 128),
    "fig3b":    Config("fig3b", 131072, 8, 32, 8, 128),
}


def _fill(draw, C: int) -> List[int]:
    """Draw lengths until the running sum reaches C; truncate the last document to fit
    (PAPER.md:224)."""
    out, total = [], 0
    while total < C:
        x = int(draw())
        x = min(x, C - total)
        out.append(x)
        total += x
    return out


def doc_lengths(name: str, seed: int = 0) -> List[int]:
    cfg = CONFIGS[name]
    rng = np.random.default_rng(seed)
    C = cfg.C
    if name == "tiny":
        return [512, 256, 128, 128]
    if name == "fig3a":
        return [131072]
    if name == "fig3b":
        return [8192] * 16
    if name == "8b":
        return _fill(lambda: np.clip(np.rint(np.exp(np.log(2048.0) + 1.0 * rng.standard_normal())),
                                     128, 32768), C)
    if name == "short":
        return _fill(lambda: rng.integers(64, 1025), C)
    if name.startswith("longtail"):
        big = C * 9 // 16                                    # 56 % of C (73728 at 128K)
        rest = _fill(lambda: np.clip(np.floor(256.0 * (1.0 - rng.random()) ** (-1.0 / 1.2)),
                                     256, C), C - big)
        pos = int(rng.integers(0, len(rest) + 1))
        return rest[:pos] + [big] + rest[pos:]
    if name == "70b":
        big_total = 78643                                    # 30 % of C
        if rng.integers(0, 2) == 0:
            bigs = [big_total]
        else:
            a = int(rng.integers(32768, big_total - 32768 + 1))
            bigs = [a, big_total - a]
        rest = _fill(lambda: np.clip(np.rint(np.exp(np.log(4096.0) + 1.0 * rng.standard_normal())),
                                     128, 32768), C - big_total)
        for b in bigs:
            pos = int(rng.integers(0, len(rest) + 1))
            rest = rest[:pos] + [b] + rest[pos:]
        return rest
    raise KeyError(name)


def random_doc_lengths(rng: np.random.Generator, C: int, lo: int, hi: int) -> List[int]:
    """Uniform lengths in [lo, hi] filled to C (used by property tests)."""
    return _fill(lambda: rng.integers(lo, hi + 1), C)


def make_tensors(C: int, Hq: int, Hkv: int, D: int, seed: int = 0, device: str = "cpu"):
    """q, k, v, dO ~ N(0,1) drawn in fp32 from a seeded generator and rounded to bf16.
    Returns torch tensors q,dO [C,Hq,D] and k,v [C,Hkv,D] on `device`."""
    import torch
    g = torch.Generator(device=device)
    g.manual_seed(seed)

    def draw(h):
        return torch.randn((C, h, D), generator=g, device=device,
                           dtype=torch.float32).to(torch.bfloat16)
    q = draw(Hq)
    k = draw(Hkv)
    v = draw(Hkv)
    do = draw(Hq)
    return q, k, v, do


def bf16_to_f64(t) -> np.ndarray:
    """Exact conversion of a bf16 torch tensor to a numpy fp64 array."""
    import torch
    return t.detach().to("cpu").to(torch.float64).numpy()
