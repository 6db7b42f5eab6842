"""Seeded weight sets for the PVFinder model of BASELINE.json config 0.

The paper's trained weights are not available (PAPER.md gives none), so two synthetic sets
stand in:

``rand``   BASELINE.json config 0 "Kaiming-uniform init", read as PyTorch's layer default
           ``kaiming_uniform_(a=sqrt(5))``: W ~ U(+-1/sqrt(fan_in)), b ~ U(+-1/sqrt(fan_in)),
           fan_in = in (Linear) or C_in*K (Conv1d).  Drawn in the order FC0..FC5, then
           e1, e2, b, d2, d1, head; W before b.
``peaky``  a hand-constructed toy vertex finder (structured signal + scaled ``rand``) whose output
           has a few well separated peaks per event, so that peak agreement is well conditioned.

Layouts are PyTorch's: Linear [out][in]; Conv1d [C_out][C_in][K]; all float32.
No method arithmetic lives here: these are inputs.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

CONV_NAMES = ("e1", "e2", "b", "d2", "d1", "head")


def fc_layer_shapes(fc_in: int = 9, hidden: int = 25, out: int = 800):
    """[(out, in)] for the six FC layers 9->25->25->25->25->25->800 (BASELINE.json config 0)."""
    dims = [fc_in] + [hidden] * 5 + [out]
    return [(dims[i + 1], dims[i]) for i in range(6)]


def unet_layer_shapes(channels: int = 64, in_ch: int = 8, kernels=(25, 15, 5, 15, 25)):
    """[(C_out, C_in, K)] for e1, e2, b, d2, d1, head (BASELINE.json config 0)."""
    C = channels
    k1, k2, kb, kd2, kd1 = kernels
    return [(C, in_ch, k1), (C, C, k2), (C, C, kb), (C, 2 * C, kd2), (C, 2 * C, kd1), (1, C, 1)]


@dataclass
class PVFWeights:
    fc_w: list = field(default_factory=list)    # 6 x float32 [out, in]
    fc_b: list = field(default_factory=list)    # 6 x float32 [out]
    conv_w: list = field(default_factory=list)  # 6 x float32 [C_out, C_in, K]  (e1,e2,b,d2,d1,head)
    conv_b: list = field(default_factory=list)  # 6 x float32 [C_out]
    channels: int = 64
    kind: str = "rand"

    def n_params(self) -> int:
        return int(sum(a.size for a in self.fc_w + self.fc_b + self.conv_w + self.conv_b))


def _uniform(rng, shape, fan_in):
    bound = 1.0 / np.sqrt(float(fan_in))
    return rng.uniform(-bound, bound, size=shape).astype(np.float32)


def _rand(seed: int, channels: int) -> PVFWeights:
    rng = np.random.default_rng(seed)
    w = PVFWeights(channels=channels, kind="rand")
    for (o, i) in fc_layer_shapes():
        w.fc_w.append(_uniform(rng, (o, i), i))
        w.fc_b.append(_uniform(rng, (o,), i))
    for (co, ci, k) in unet_layer_shapes(channels):
        w.conv_w.append(_uniform(rng, (co, ci, k), ci * k))
        w.conv_b.append(_uniform(rng, (co,), ci * k))
    return w


def _peaky(seed: int, channels: int, eps_unet: float = 0.3, eps_fc: float = 0.01,
           head_gain: float = 0.16, head_bias: float = -6.5) -> PVFWeights:
    C = channels
    noise = _rand(seed, channels)
    w = PVFWeights(channels=channels, kind="peaky")
    fcs = fc_layer_shapes()
    # FC0: 24 hinges on feature 0 (z relative to the interval edge) + one constant unit.
    knots = -0.05 + np.arange(24) * (1.10 / 23.0)
    W0 = np.zeros(fcs[0], np.float64)
    b0 = np.zeros(fcs[0][0], np.float64)
    W0[:24, 0] = 1.0
    b0[:24] = -knots
    b0[24] = 1.0
    S_w = [W0]
    S_b = [b0]
    for _ in range(4):  # FC1..FC4: identity
        S_w.append(np.eye(25))
        S_b.append(np.zeros(25))
    # FC5: piecewise-linear interpolant (on the hinge knots) of a Gaussian bump per output bin.
    c_idx = np.repeat(np.arange(8), 100)
    l_idx = np.tile(np.arange(100), 8)
    u_l = (l_idx + 0.5) / 100.0
    s_c = (4.0 + c_idx) / 100.0
    g = 5.54 * np.exp(-(knots[None, :] - u_l[:, None]) ** 2 / (2.0 * s_c[:, None] ** 2)) - 5.0  # [800,24]
    slope = np.diff(g, axis=1) / np.diff(knots)[None, :]                                       # [800,23]
    W5 = np.zeros(fcs[5], np.float64)
    W5[:, 0] = slope[:, 0]
    W5[:, 1:23] = slope[:, 1:] - slope[:, :-1]
    W5[:, 23] = -slope[:, -1]          # flat after the last knot
    W5[:, 24] = g[:, 0]
    S_w.append(W5)
    S_b.append(np.zeros(800))
    for k in range(6):
        w.fc_w.append((S_w[k] + eps_fc * noise.fc_w[k]).astype(np.float32))
        w.fc_b.append((S_b[k] + eps_fc * noise.fc_b[k]).astype(np.float32))
    # UNet: smooth channel 0 in e1, pass it through the first skip channel of d1, read it in the head.
    shapes = unet_layer_shapes(C)
    S_cw = [np.zeros(s, np.float64) for s in shapes]
    S_cb = [np.zeros(s[0], np.float64) for s in shapes]
    k1 = shapes[0][2]
    taps = np.exp(-0.5 * ((np.arange(k1) - (k1 - 1) / 2.0) / 1.5) ** 2)
    S_cw[0][0, 0, :] = taps / taps.sum()
    kd1 = shapes[4][2]
    S_cw[4][0, C + 0, (kd1 - 1) // 2] = 1.0   # concat order is [upsampled, skip]
    # head: background logit -6.5 (p = 1.5e-3, a decade below the 0.01 peak threshold, so that ripples of
    # the background are not peaks: DESIGN.md "peaky weights"), signal gain 0.16
    # (head_gain / head_bias are parameters only so that tests/test_oracle_pins.py can re-run the conditioning
    # experiment that compares this recipe with the first one, gain 0.12 / bias -5)
    S_cw[5][0, 0, 0] = head_gain
    S_cb[5][0] = head_bias
    for k in range(6):
        w.conv_w.append((S_cw[k] + eps_unet * noise.conv_w[k]).astype(np.float32))
        w.conv_b.append((S_cb[k] + eps_unet * noise.conv_b[k]).astype(np.float32))
    return w


def make_weights(kind: str, seed: int, channels: int = 64, **peaky_kw) -> PVFWeights:
    if kind == "rand":
        return _rand(seed, channels)
    if kind == "peaky":
        return _peaky(seed, channels, **peaky_kw)
    raise ValueError(f"unknown weight kind {kind!r}")
