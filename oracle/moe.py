"""O8 extended to mixture-of-experts layers.  Test oracle.

The paper evaluates Qwen3-MoE 30B with the same mechanism; a sparse MLP has one more function-preserving
symmetry than a dense one: the ORDER of the experts, as long as the router's rows move with them.  Readings (recorded in
DESIGN.md): weights in Linear convention, router [E, H], gate/up [E, I, H], down [E, H, I];

  (eps, _) = keygen(key, EXPERT|layer, E)                  new expert e' is old expert eps[e']
      router'[e', :] = router[eps[e'], :]
  for every OLD expert e:  (pi_e, _) = keygen(key, EXPERT_MLP|(layer*E + e), I)       its own neuron permutation
      gate'[e'] = gate[eps[e']][pi_e, :]   up'[e'] = up[eps[e']][pi_e, :]   down'[e'] = down[eps[e']][:, pi_e]   (e = eps[e'])

  MoE(x) = sum over the top-k experts e of  softmax_topk(logits)_e * MLP_e(x),   logits = router . x,
  top-k by logit, ties to the smaller index (the usual sparse-MoE forward; no shared expert, no bias).
Permuting experts relabels them and permutes the logits the same way, so the selected set, the weights and every
expert's output are unchanged: MoE' = MoE up to fp reassociation (ties in the logits aside: measure zero).
"""
import numpy as np
from .keygen import keygen
from .linear import to_f64, silu


def stream_expert(layer):
    return (7 << 32) | layer


def stream_expert_mlp(layer, n_experts, e):
    return (8 << 32) | (layer * n_experts + e)


def expert_perm(key, layer, n_experts):
    return keygen(key, stream_expert(layer), n_experts)[0]


def expert_mlp_perm(key, layer, n_experts, e, inter):
    return keygen(key, stream_expert_mlp(layer, n_experts, e), inter)[0]


def permute_experts(router, gate, up, down, eps, pis):
    """router [E, H], gate/up [E, I, H], down [E, H, I] (any dtype); eps [E]; pis[e] = neuron permutation of OLD expert e."""
    E = router.shape[0]
    r2, g2, u2, d2 = (np.empty_like(a) for a in (router, gate, up, down))
    for en in range(E):
        e = int(eps[en])
        pi = np.asarray(pis[e], dtype=np.int64)
        r2[en] = router[e]
        g2[en] = gate[e][pi, :]
        u2[en] = up[e][pi, :]
        d2[en] = down[e][:, pi]
    return r2, g2, u2, d2


def topk_experts(logits, k):
    """Indices of the k largest logits of one token, ties to the smaller index, in descending order of logit."""
    order = sorted(range(len(logits)), key=lambda e: (-float(logits[e]), e))
    return order[:k]


def moe_f64(x, router, gate, up, down, k):
    """x [tokens, H] -> [tokens, H], fp64 throughout."""
    x, router = to_f64(x), to_f64(router)
    out = np.zeros((x.shape[0], down.shape[1]), dtype=np.float64)
    logits = x @ router.T
    for t in range(x.shape[0]):
        sel = topk_experts(logits[t], k)
        z = logits[t, sel]
        w = np.exp(z - z.max())
        w /= w.sum()
        for wi, e in zip(w, sel):
            g = to_f64(gate[e]) @ x[t]
            u = to_f64(up[e]) @ x[t]
            out[t] += wi * (to_f64(down[e]) @ (silu(g) * u))
    return out
