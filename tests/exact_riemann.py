"""Exact self-similar solution of the 1D relativistic Riemann problem for p = cs^2 e (pin P8).

Textbook closed form (simple rarefaction wave + Taub jump conditions), NOT from the paper and
NOT from oracle/: it is what the assembled oracle is pinned against (P8).
  fan:      v = (xi + cs)/(1 + xi cs),  e = eL ((1-v)/(1+v))^kappa,  kappa = (1+cs^2)/(2 cs)
  plateau:  v* = (1-a)/(1+a), a = (e*/eL)^(1/kappa)   [Riemann invariant]
            v*^2 = 3 (e*-eR)^2 / ((3e*+eR)(3eR+e*))   [Taub, cs^2 = 1/3]
  shock:    vsh^2 = (3e*+eR)/(3(3eR+e*))
  contact at xi = v*: only n jumps.
"""
import numpy as np
from scipy.optimize import brentq

CS = 1.0 / np.sqrt(3.0)
KAPPA = (1.0 + CS * CS) / (2.0 * CS)


def plateau(eL, eR):
    def g(es):
        a = (es / eL) ** (1.0 / KAPPA)
        v_r = (1.0 - a) / (1.0 + a)
        v_s = np.sqrt(3.0 * (es - eR) ** 2 / ((3.0 * es + eR) * (3.0 * eR + es)))
        return v_r - v_s
    es = brentq(g, eR * (1 + 1e-12), eL * (1 - 1e-12), xtol=1e-300, rtol=1e-14)
    a = (es / eL) ** (1.0 / KAPPA)
    vs = (1.0 - a) / (1.0 + a)
    vsh = np.sqrt((3.0 * es + eR) / (3.0 * (3.0 * eR + es)))
    xi_t = (vs - CS) / (1.0 - vs * CS)
    return es, vs, vsh, xi_t


def solution(xi, eL, eR, nL=None, nR=None):
    """returns e(xi), v(xi), n(xi)"""
    nL = eL ** 0.75 if nL is None else nL
    nR = eR ** 0.75 if nR is None else nR
    es, vs, vsh, xi_t = plateau(eL, eR)
    xi = np.asarray(xi, dtype=np.float64)
    e = np.empty_like(xi); v = np.empty_like(xi); n = np.empty_like(xi)
    left = xi <= -CS
    fan = (xi > -CS) & (xi <= xi_t)
    plat_l = (xi > xi_t) & (xi <= vs)
    plat_r = (xi > vs) & (xi <= vsh)
    right = xi > vsh
    e[left], v[left], n[left] = eL, 0.0, nL
    vf = (xi[fan] + CS) / (1.0 + xi[fan] * CS)
    ef = eL * ((1.0 - vf) / (1.0 + vf)) ** KAPPA
    e[fan], v[fan], n[fan] = ef, vf, nL * (ef / eL) ** 0.75
    gs = 1.0 / np.sqrt(1.0 - vs * vs)
    e[plat_l], v[plat_l], n[plat_l] = es, vs, nL * (es / eL) ** 0.75
    e[plat_r], v[plat_r], n[plat_r] = es, vs, nR * vsh / (gs * (vsh - vs))
    e[right], v[right], n[right] = eR, 0.0, nR
    return e, v, n
