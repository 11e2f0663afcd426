"""Brute-force enumeration of the 2x2x2 periodic RFIM (256 states), written with numpy only.

Independent of oracle/: H(s) = -J sum_<ij> s_i s_j - hs sum_i f_i s_i (Eq. 1) with the
3N directed bonds (i,i+x),(i,i+y),(i,i+z); on L=2 the +1 and -1 neighbour coincide, so every
distinct pair is counted twice -- the same convention the six-neighbour sum uses.
"""
import numpy as np


def all_states():
    """int8 [256, 8] of +-1, site index i = x + 2*(y + 2*z)."""
    codes = np.arange(256)
    bits = (codes[:, None] >> np.arange(8)[None, :]) & 1
    return (2 * bits - 1).astype(np.int64)


def hamiltonian(states, J, hs, field):
    s = states.reshape(-1, 2, 2, 2)            # [state, z, y, x]
    eb = (s * (np.roll(s, -1, axis=3) + np.roll(s, -1, axis=2) + np.roll(s, -1, axis=1))).sum(axis=(1, 2, 3))
    ef = (states * np.asarray(field, dtype=np.float64)[None, :]).sum(axis=1)
    return -J * eb - hs * ef


def boltzmann(states, J, hs, field, T):
    H = hamiltonian(states, J, hs, field)
    w = np.exp(-(H - H.min()) / T)
    return H, w / w.sum()


def exact_averages(J, hs, field, T):
    st = all_states()
    H, p = boltzmann(st, J, hs, field, T)
    m = st.sum(axis=1) / 8.0
    return float((p * H).sum()), float((p * np.abs(m)).sum())


def exact_moments(J, hs, field, T):
    """Exact <e>, <e^2>, <|m|>, <m^2>, <m^4> of the 2x2x2 lattice (e = H/8 per site, m = mean spin)."""
    st = all_states()
    H, p = boltzmann(st, J, hs, field, T)
    e = H / 8.0
    m = st.sum(axis=1) / 8.0
    return np.array([(p * e).sum(), (p * e * e).sum(), (p * np.abs(m)).sum(), (p * m ** 2).sum(), (p * m ** 4).sum()])
