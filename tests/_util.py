"""Helpers shared by the GPU parity tests (marshalling and comparison only; no method arithmetic)."""
import numpy as np
import torch

import oracle
from paper_2607_07494_b200 import gf8, synth


def relfro(a, b):
    a, b = np.asarray(a, np.float64), np.asarray(b, np.float64)
    return float(np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300))


def code_ordinal(codes):
    """Signed position of each FP8 code on the number line (+0 and -0 both map to 0)."""
    c = np.asarray(codes).astype(np.int32)
    mag = c & 0x7F
    return np.where(c & 0x80, -mag, mag)


def code_mismatch(gpu_codes, orc_codes):
    """(fraction of differing elements, largest distance in code steps)."""
    d = np.abs(code_ordinal(gpu_codes) - code_ordinal(orc_codes))
    return float((d > 0).mean()), int(d.max())


def to_np64(t):
    return t.detach().double().cpu().numpy()


def bf16_bits(t):
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16)


def bf16_ordinal(bits):
    b = bits.astype(np.int32)
    mag = b & 0x7FFF
    return np.where(b & 0x8000, -mag, mag)


class Case:
    """One gradient matrix with its factors, oracle bases and a gf8 context holding the same bases."""

    def __init__(self, m, n, kG, kA, side, dtype, seed, T=None, fmt=gf8.E4M3, scaling=gf8.SCALE_TENSOR,
                 damping=1e-3, q=4, precision=gf8.PREC_EXACT, device="cuda"):
        self.m, self.n, self.kG, self.kA, self.side = m, n, kG, kA, side
        self.fmt, self.scaling, self.damping = fmt, scaling, damping
        self.tdtype = torch.bfloat16 if dtype == "bf16" else torch.float32
        T = T or 2 * max(m, n)
        useA, useG = bool(side & gf8.SIDE_IN), bool(side & gf8.SIDE_OUT)
        G = synth.gradient(m, n, device, seed, 0)
        self.G = G.to(self.tdtype)
        self.X = synth.factor_samples(T, n, device, seed, 1).to(self.tdtype) if useA else None
        self.D = synth.factor_samples(T, m, device, seed, 2).to(self.tdtype) if useG else None
        self.V0A = synth.start_basis(n, kA, device, seed, 3) if useA else None
        self.V0G = synth.start_basis(m, kG, device, seed, 4) if useG else None
        # oracle state
        self.A = oracle.factor_accumulate(to_np64(self.X)) if useA else None
        self.Gf = oracle.factor_accumulate(to_np64(self.D)) if useG else None
        self.bA = oracle.refresh_basis(self.A, to_np64(self.V0A), q, damping) if useA else None
        self.bG = oracle.refresh_basis(self.Gf, to_np64(self.V0G), q, damping) if useG else None
        self.layer = gf8.Layer(m, n, side, kA if useA else 0, kG if useG else 0, fmt, scaling, damping, 0.0)
        self.ctx = gf8.create([self.layer], precision)
        self.hand_over_bases()

    def hand_over_bases(self):
        dev = self.G.device
        for side, b in ((gf8.SIDE_IN, self.bA), (gf8.SIDE_OUT, self.bG)):
            if b is not None:
                self.ctx.set_basis(0, side, torch.from_numpy(b.U).float().to(dev).contiguous(),
                                   torch.from_numpy(b.mu).float().to(dev).contiguous(), float(b.rho))

    def rank_grad(self, r):
        return synth.rank_gradient(self.G, r, 99).to(self.tdtype)

    def oracle_encode(self, g):
        return oracle.encode(to_np64(g), self.bG, self.bA, self.fmt, self.scaling)

    def oracle_reduce_decoded(self, codes, sinvs, average=True):
        return oracle.reduce_decoded(codes, sinvs, self.bG, self.bA, self.fmt, self.scaling, average)
