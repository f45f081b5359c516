"""O8 -- function-preserving neuron / attention-head permutation.  Test oracle.

The paper names "inter- and intra-layer weight shuffling" (abstract) and "randomizing both
virtual-to-physical mappings and tensor layout" (Figure 3 caption) and says nothing more.
BJ:north_star (b) gives it meaning: "an intra-layer neuron permutation that preserves the function
(rows of W_gate/W_up and columns of W_down, and whole attention heads, permuted together)".
Reading O8 of SURVEY.md (weights in Linear convention [out, in], row-major):

  MLP, I = intermediate:  (pi, _) = keygen(key, MLP|layer, I)
      gate'[r, :] = gate[pi[r], :]    up'[r, :] = up[pi[r], :]    down'[:, r] = down[:, pi[r]]
  Heads, G = n_q / n_kv, d = head_dim:
      (kappa, _) = keygen(key, KVHEAD|layer, n_kv)
      for each new group g':  (rho_g', _) = keygen(key, QGROUP|(layer*n_kv + g'), G)
      new q head h' = g'*G + j' takes old q head eta[h'] = kappa[g']*G + rho_g'[j']
      k', v' row-groups of d rows move by kappa; q' row-groups by eta; o' column-groups by eta.
  Elements inside a head are not reordered.  MHA is G = 1.
"""
import numpy as np
from .keygen import keygen, stream_mlp, stream_kvhead, stream_qgroup


def mlp_perm(key, layer, inter):
    return keygen(key, stream_mlp(layer), inter)[0]


def head_maps(key, layer, n_q, n_kv):
    """(kappa [n_kv], eta [n_q]) of O8."""
    if n_q % n_kv:
        raise ValueError("n_q must be a multiple of n_kv")
    G = n_q // n_kv
    kappa = keygen(key, stream_kvhead(layer), n_kv)[0]
    eta = np.empty(n_q, dtype=np.uint32)
    for g in range(n_kv):
        rho = keygen(key, stream_qgroup(layer, n_kv, g), G)[0]
        for j in range(G):
            eta[g * G + j] = int(kappa[g]) * G + int(rho[j])
    return kappa, eta


def expand_head_rows(head_map, d):
    """Row (or column) index map for whole heads: new index h'*d + c takes old head_map[h']*d + c."""
    hm = np.asarray(head_map, dtype=np.int64)
    return (hm[:, None] * d + np.arange(d, dtype=np.int64)[None, :]).ravel()


def permute_mlp(gate, up, down, pi):
    """Arrays of any dtype, shapes gate/up [I, H], down [H, I]."""
    pi = np.asarray(pi, dtype=np.int64)
    return gate[pi, :].copy(), up[pi, :].copy(), down[:, pi].copy()


def permute_heads(q, k, v, o, kappa, eta, d):
    """q [n_q*d, H], k/v [n_kv*d, H], o [H, n_q*d]."""
    rq = expand_head_rows(eta, d)
    rk = expand_head_rows(kappa, d)
    return q[rq, :].copy(), k[rk, :].copy(), v[rk, :].copy(), o[:, rq].copy()
