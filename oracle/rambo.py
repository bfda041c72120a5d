"""ORACLE (test infrastructure, NOT the product): seeded synthetic inputs, counter-based PRNG + RAMBO flat phase space.

Plain numpy restatement of steps 1-2 of the MC chain ("random numbers are drawn ... converted into particle
momenta using a phase space sampling algorithm"; the paper's standalone application does both
data-parallel).  Two roles:
  * it writes the seeded input buffers (momenta, g_s, r_hel, r_col) that the oracle tests and the GPU parity tests
    feed to both sides; it holds none of the matrix-element arithmetic;
  * it is the oracle of the product's device-side generator me_generate (csrc/me_rambo.cu):
    tests/test_gpu_rambo.py compares the two (uniforms bit-exact, momenta and weights to rounding).  Each side
    implements the same counter-based generator on its own (splitmix64 steps); they share no code.
Pinned by tests/test_inputs.py (P15: closed-form weights, N = 2 and N = 3 phase-space volumes, momentum conservation,
mass shells, stream independence).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / reference legs
import it; bench.py's GPU arm makes its inputs with me_generate.  numpy only; no torch, no CUDA.

Recipe: sqrt(s) = 1500 GeV, incoming p0 = (E,0,0,+E),
p1 = (E,0,0,-E), final state from RAMBO (massless generation -> conformal boost to the CM frame ->
xi-rescaling by Newton iteration for masses), 4 uniforms per final-state particle, no cuts.
Independent streams for momenta, alpha_s, r_hel, r_col.
"""
from __future__ import annotations

import math

import numpy as np

# stream ids (independent counter spaces)
STREAM_MOMENTA = 0
STREAM_ALPHAS = 1
STREAM_RNDHEL = 2
STREAM_RNDCOL = 3

# process table: name -> (npar, final-state masses as multiples of mt: 1 = top, 0 = massless)
PROCESSES = {
    "ee_mumu": dict(npar=4, final_top=(0, 0), ngluon=0),
    "gg_tt": dict(npar=4, final_top=(1, 1), ngluon=2),
    "gg_ttg": dict(npar=5, final_top=(1, 1, 0), ngluon=3),
    "gg_ttgg": dict(npar=6, final_top=(1, 1, 0, 0), ngluon=4),
    "gg_ttggg": dict(npar=7, final_top=(1, 1, 0, 0, 0), ngluon=5),
    # g ubar -> tau+ tau- + (n-1) g + ubar, all massless (Table 4 is n = 3)
    "gux_taptamux": dict(npar=5, final_top=(0, 0, 0), ngluon=1),
    "gux_taptamgux": dict(npar=6, final_top=(0, 0, 0, 0), ngluon=2),
    "gux_taptamggux": dict(npar=7, final_top=(0, 0, 0, 0, 0), ngluon=3),
}

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(x: np.ndarray) -> np.ndarray:
    """One splitmix64 output step applied elementwise to uint64 state x (wraps mod 2^64)."""
    with np.errstate(over="ignore"):
        z = x + np.uint64(0x9E3779B97F4A7C15)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def uniforms(seed: int, stream: int, start: int, count: int) -> np.ndarray:
    """count uniforms in (0,1), a pure function of (seed, stream, index): index = start..start+count-1.

    u = (top 53 bits + 0.5) / 2^53, so 0 < u < 1 strictly (log(u) is always finite).
    """
    idx = np.arange(start, start + count, dtype=np.uint64)
    with np.errstate(over="ignore"):
        key = _splitmix64(np.uint64(seed) * np.uint64(0xD1342543DE82EF95) + np.uint64(stream + 1))
        x = _splitmix64(idx ^ key)
        x = _splitmix64(x + key)
    return ((x >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def rambo(r: np.ndarray, masses, w: float):
    """RAMBO (Kleiss, Stirling, Ellis 1986).  r: [nevt][N][4] uniforms; masses: N floats; w = sqrt(s).

    Returns (p [nevt][N][4] as (E,px,py,pz), weight [nevt]) with the Lorentz-invariant phase-space
    weight in the convention dPhi_N = prod d^3p/((2pi)^3 2E) (2pi)^4 delta^4.
    """
    r = np.asarray(r, dtype=np.float64)
    nevt, n, _ = r.shape
    masses = np.asarray(masses, dtype=np.float64)
    c = 2.0 * r[:, :, 0] - 1.0
    s = np.sqrt(1.0 - c * c)
    phi = 2.0 * math.pi * r[:, :, 1]
    f = -np.log(r[:, :, 2] * r[:, :, 3])
    q = np.stack([f, f * s * np.cos(phi), f * s * np.sin(phi), f * c], axis=-1)
    qs = q.sum(axis=1)  # [nevt][4]
    mq = np.sqrt(qs[:, 0] ** 2 - qs[:, 1] ** 2 - qs[:, 2] ** 2 - qs[:, 3] ** 2)
    b = -qs[:, 1:] / mq[:, None]
    x = w / mq
    g = qs[:, 0] / mq
    a = 1.0 / (1.0 + g)
    bq = np.einsum("ej,enj->en", b, q[:, :, 1:])
    p = np.empty_like(q)
    p[:, :, 0] = x[:, None] * (g[:, None] * q[:, :, 0] + bq)
    p[:, :, 1:] = x[:, None, None] * (
        q[:, :, 1:] + b[:, None, :] * q[:, :, 0:1] + (a[:, None] * bq)[:, :, None] * b[:, None, :]
    )
    # massless weight
    wt0 = (
        (math.pi / 2.0) ** (n - 1)
        * w ** (2 * n - 4)
        / (math.factorial(n - 1) * math.factorial(n - 2))
        * (2.0 * math.pi) ** (4 - 3 * n)
    )
    wt = np.full(nevt, wt0)
    if np.any(masses != 0.0):
        m2 = masses**2
        e0 = p[:, :, 0]
        xi = np.full(nevt, math.sqrt(1.0 - (masses.sum() / w) ** 2))
        for _ in range(50):
            e = np.sqrt(m2[None, :] + (xi**2)[:, None] * e0**2)
            f0 = e.sum(axis=1) - w
            g0 = (xi[:, None] * e0**2 / e).sum(axis=1)
            dxi = f0 / g0
            xi = xi - dxi
            if np.max(np.abs(dxi)) < 1e-15:
                break
        e = np.sqrt(m2[None, :] + (xi**2)[:, None] * e0**2)
        k = xi[:, None] * e0  # |p| after rescaling
        p[:, :, 1:] *= xi[:, None, None]
        p[:, :, 0] = e
        wt = wt * (k.sum(axis=1) / w) ** (2 * n - 3) * np.prod(k / e, axis=1) * w / (k * k / e).sum(axis=1)
    return p, wt


def make_momenta(process: str, nevt: int, seed: int = 1, sqrts: float = 1500.0, mt: float = 173.0,
                 start: int = 0, return_weight: bool = False):
    """momenta[nevt][npar][4] (E,px,py,pz) in GeV for events start..start+nevt-1 of the seeded stream."""
    info = PROCESSES[process]
    npar = info["npar"]
    nfin = npar - 2
    masses = [mt * t for t in info["final_top"]]
    r = uniforms(seed, STREAM_MOMENTA, start * nfin * 4, nevt * nfin * 4).reshape(nevt, nfin, 4)
    pf, wt = rambo(r, masses, sqrts)
    p = np.empty((nevt, npar, 4), dtype=np.float64)
    e = 0.5 * sqrts
    p[:, 0, :] = (e, 0.0, 0.0, e)
    p[:, 1, :] = (e, 0.0, 0.0, -e)
    p[:, 2:, :] = pf
    return (p, wt) if return_weight else p


def make_gs(nevt: int, seed: int = 1, alphas=None, start: int = 0) -> np.ndarray:
    """g_s = sqrt(4 pi alpha_s) per event.  alphas = float: fixed; None: alpha_s ~ U[0.10, 0.13] (BASELINE config 4)."""
    if alphas is not None:
        return np.full(nevt, math.sqrt(4.0 * math.pi * alphas))
    u = uniforms(seed, STREAM_ALPHAS, start, nevt)
    return np.sqrt(4.0 * math.pi * (0.10 + 0.03 * u))


def make_rnd(nevt: int, seed: int = 1, start: int = 0):
    """(r_hel, r_col): two independent uniform streams in (0,1), one value per event."""
    return uniforms(seed, STREAM_RNDHEL, start, nevt), uniforms(seed, STREAM_RNDCOL, start, nevt)


def lorentz_transform(p: np.ndarray, seed: int = 7) -> np.ndarray:
    """Apply one random rotation followed by one random boost (|beta| <= 0.6) to all momenta of each event."""
    p = np.asarray(p, dtype=np.float64)
    nevt = p.shape[0]
    u = uniforms(seed, 17, 0, nevt * 7).reshape(nevt, 7)
    # random unit quaternion -> rotation matrix
    qn = u[:, :4] - 0.5
    qn /= np.linalg.norm(qn, axis=1, keepdims=True)
    a, b, c, d = qn.T
    rot = np.stack([
        np.stack([a * a + b * b - c * c - d * d, 2 * (b * c - a * d), 2 * (b * d + a * c)], -1),
        np.stack([2 * (b * c + a * d), a * a - b * b + c * c - d * d, 2 * (c * d - a * b)], -1),
        np.stack([2 * (b * d - a * c), 2 * (c * d + a * b), a * a - b * b - c * c + d * d], -1),
    ], 1)
    beta = (u[:, 4:7] - 0.5) * (1.2 / math.sqrt(3.0))
    b2 = (beta**2).sum(1)
    gam = 1.0 / np.sqrt(1.0 - b2)
    out = np.empty_like(p)
    pv = np.einsum("eij,enj->eni", rot, p[:, :, 1:])
    bp = np.einsum("ej,enj->en", beta, pv)
    e = p[:, :, 0]
    out[:, :, 0] = gam[:, None] * (e + bp)
    coef = ((gam - 1.0) / np.where(b2 > 0, b2, 1.0))[:, None] * bp + gam[:, None] * e
    out[:, :, 1:] = pv + coef[:, :, None] * beta[:, None, :]
    return out
