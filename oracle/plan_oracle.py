"""Oracle for the planner / cost model (``osdp_cost_eval``, ``osdp_plan``).  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s baseline legs may import this file.
It shares no code with ``paper_2305_09940_b200/csrc`` and imports nothing from that package.

Follows the paper step by step:

* Memory cost M_i (§3.1):  DP: M_model + b M_act + M_extra;  ZDP: M_model/N + b M_act + M_extra.
  With operator splitting the split part goes size -> size / slice_granularity, applied to
  the sliceable part of M_extra (reading P1).  Slices are "released serially", so a
  transient workspace is live for one operator at a time: reading P6 keeps both accountings,
      M(p) = sum_i [ model_i/(N or 1) + b act_i + extra_fixed_i + ceil(extra_summed_i / k_i) ]
             + max_i ceil(extra_transient_i / k_i).
  k = 1 and extra_transient = 0 give the paper's formula exactly.
* Time cost T_i:  c_p (N-1)(alpha + S_i beta / N) + b gamma_i,  c_DP = 2, c_ZDP = 3,
  plus (k-1) delta_i, our per-extra-slice overhead (reading P2; delta = 0 is the paper's model).
* Search (Algorithm 1 lines 5-11; b fixed, reading P3): traverse every plan, keep the
  feasible plan with strictly smaller time ("<", line 8).  Options per operator are ordered DP before
  ZDP and k ascending in the caller's candidate list; plans are traversed in lexicographic order of
  option indices, so among equal-time optima the first (least split, DP-most) wins (reading P5).
  Where floating point decides this integer outcome both sides take the decision in the same precision
  (reading P9): every T_i is rounded once to an integer count of picoseconds, floor(T_i * 1e12 + 0.5),
  and plan times are exact integer sums of those.
* Infeasible (Algorithm 1 lines 12-14): returns None.
* Slice-level mode mixing (reading P10): cost_eval_mixed / plan_brute_force_mixed.
* Batch loop (Algorithm 1 lines 3-20, reading f3): b = 1, 2, 3, ...; stop at the first b with no feasible
  plan; return the candidate minimising T(b)/b (Eq. 1's objective is the per-sample time).

Pins (tests/test_planner.py): closed forms the paper states — ZDP/DP communication ratio 3/2
(PAPER.md:25,47,94), model-state memory 1/N, N = 1 => modes coincide, sliceable term
~ 1/k, 0.6e9 params x 4 B = 2.24 GiB, M_limit = inf => all DP / k = 1,
M_limit below the minimum => infeasible, monotonicity in M_limit.
"""
from __future__ import annotations

import dataclasses
import itertools
import math

DP, ZDP = 0, 1


@dataclasses.dataclass
class OpCost:
    S: float = 0.0                 # parameter bytes moved by one collective (S_i)
    model: int = 0                 # M_i^(model) bytes
    act: int = 0                   # M_i^(act) bytes per unit batch
    extra_fixed: int = 0           # M_i^(extra), part that splitting does not shrink
    extra_summed: int = 0          # M_i^(extra), sliceable, summed over operators (paper's Eq. 1 sum)
    extra_transient: int = 0       # M_i^(extra), sliceable, live for one operator at a time
    gamma: float = 0.0             # seconds per unit batch
    delta: float = 0.0             # seconds per extra slice


@dataclasses.dataclass
class Device:
    N: int = 1
    alpha: float = 0.0
    beta: float = 0.0
    mem_limit: int = 0
    # Activation checkpointing ("about 30% extra computation overhead"; "the recomputation
    # process before backward propagation requires an additional round of gathering"; reading P12).  Off = the paper's
    # plain cost model.
    checkpointing: bool = False
    recompute_fraction: float = 0.0
    act_keep_fraction: float = 1.0


def ceil_div(a: int, b: int) -> int:
    return -(-a // b)


def cost_eval(op: OpCost, mode: int, k: int, b: int, dev: Device):
    """(persistent_bytes, transient_bytes, seconds) of one operator under (mode, k, b)."""
    model = ceil_div(op.model, dev.N) if mode == ZDP else op.model
    persist = model + _act_bytes(op, b, dev) + op.extra_fixed + ceil_div(op.extra_summed, k)
    transient = ceil_div(op.extra_transient, k)
    c = (4.0 if dev.checkpointing else 3.0) if mode == ZDP else 2.0
    t = c * (dev.N - 1) * (dev.alpha + op.S * dev.beta / dev.N) + _compute_seconds(op, b, dev) + (k - 1) * op.delta
    return persist, transient, t


def _act_bytes(op: OpCost, b: int, dev: Device) -> int:
    """b M_act, of which only the checkpoints stay resident under activation checkpointing."""
    return math.ceil(b * op.act * dev.act_keep_fraction) if dev.checkpointing else b * op.act


def _compute_seconds(op: OpCost, b: int, dev: Device) -> float:
    """b gamma, plus the recomputation of the forward under activation checkpointing."""
    return b * op.gamma * (1.0 + dev.recompute_fraction) if dev.checkpointing else b * op.gamma


def to_ps(seconds: float) -> int:
    return int(math.floor(seconds * 1e12 + 0.5))


def plan_memory_time(ops, modes, ks, b, dev):
    """(peak bytes, integer picoseconds) of a whole plan."""
    tot, tr, t = 0, 0, 0
    for op, m, k in zip(ops, modes, ks):
        p, x, ti = cost_eval(op, m, k, b, dev)
        tot += p
        tr = max(tr, x)
        t += to_ps(ti)
    return tot + tr, t


def plan_brute_force(ops, dev: Device, b: int, k_candidates):
    """Algorithm 1 lines 4-11 for one batch size: full enumeration, strict '<'.

    Returns (modes, ks, picoseconds, peak_bytes) or None when no plan fits.
    """
    options = [(m, k) for m in (DP, ZDP) for k in k_candidates]
    best = None
    best_t = math.inf
    for choice in itertools.product(range(len(options)), repeat=len(ops)):
        modes = [options[c][0] for c in choice]
        ks = [options[c][1] for c in choice]
        mem, t = plan_memory_time(ops, modes, ks, b, dev)
        if mem <= dev.mem_limit and t < best_t:
            best_t = t
            best = (modes, ks, t, mem)
    return best


# ----- slice-level mode mixing (reading P10) --------------------------------------------------
def cost_eval_mixed(op: OpCost, k: int, z: int, b: int, dev: Device):
    """An operator partitioned into k slices, z of them processed in ZDP mode and k - z in DP mode ("partition the
    operator into 4 slices and process 1 of them in the ZDP mode and 3 of them in the DP mode").
    Every slice holds 1/k of the model states and moves 1/k of the parameters: the ZDP slices' share of the model
    states, ceil(model z / k), is divided by N, the rest is replicated; a DP slice costs
    2 collectives over its S/k bytes and a ZDP slice 3, with the latency term alpha shared in the
    same proportion, so the operator's factor is (2 (k - z) + 3 z) / k = 2 + z / k."""
    assert 0 <= z <= k
    zdp_share = ceil_div(op.model * z, k)
    model = (op.model - zdp_share) + ceil_div(zdp_share, dev.N)
    persist = model + _act_bytes(op, b, dev) + op.extra_fixed + ceil_div(op.extra_summed, k)
    transient = ceil_div(op.extra_transient, k)
    c = (2.0 * (k - z) + (4.0 if dev.checkpointing else 3.0) * z) / k
    t = c * (dev.N - 1) * (dev.alpha + op.S * dev.beta / dev.N) + _compute_seconds(op, b, dev) + (k - 1) * op.delta
    return persist, transient, t


def plan_brute_force_mixed(ops, dev: Device, b: int, k_candidates):
    """Full enumeration over (k, z) per operator, k ascending then z ascending, strict '<' (first optimum wins).
    Returns (ks, zs, picoseconds, peak_bytes) or None."""
    options = [(k, z) for k in k_candidates for z in range(k + 1)]
    best, best_t = None, math.inf
    for choice in itertools.product(range(len(options)), repeat=len(ops)):
        tot, tr, t = 0, 0, 0
        for op, c in zip(ops, choice):
            p, x, ti = cost_eval_mixed(op, options[c][0], options[c][1], b, dev)
            tot += p
            tr = max(tr, x)
            t += to_ps(ti)
        if tot + tr <= dev.mem_limit and t < best_t:
            best_t = t
            best = ([options[c][0] for c in choice], [options[c][1] for c in choice], t, tot + tr)
    return best


def schedule_brute_force(ops, dev: Device, k_candidates, b_max: int = 1 << 20):
    """Algorithm 1 in full: returns (modes, ks, picoseconds, peak_bytes, b) minimising time / b, or None."""
    cands = []
    b = 1
    while b <= b_max:
        r = plan_brute_force(ops, dev, b, k_candidates)
        if r is None:
            break
        cands.append(r + (b,))
        b += 1
    if not cands:
        return None
    best = None
    for c in cands:
        if best is None or c[2] * best[4] < best[2] * c[4]:      # T(b)/b, exact integer comparison
            best = c
    return best


# ----- factor calculator for the MLP operator of this build ("calculated according to the
# definition of operators (e.g., types and shapes)"); written from DESIGN.md "Cost model", not from the
# library source. -------------------------------------------------------------------------------------
def mlp_workspace_bytes(T: int, h: int, f: int, e: int, k: int, backward: bool) -> int:
    """Bytes of per-slice tensors one call keeps beside the caller's tensors - what PAPER.md:167 fixes ("the extra
    memory required for one slice is size / slice_granularity") and SURVEY.md section 8(d) prints: one T_s x f tensor
    forward (H_s), two backward (Z_s / dZ_s and H_s), T_s = ceil(T / k), each rounded up to 256 B.  Nothing else: any
    scratch an implementation adds on top (partial sums of the bias gradients, synchronisation words) is ITS choice,
    not the method's, so it is not stated here; the tests bound it instead (reading W1)."""
    Ts = ceil_div(T, k)
    buf = ceil_div(Ts * f * e, 256) * 256
    return 2 * buf if backward else buf


def mlp_persistent_bytes(T: int, h: int, f: int, e: int, backward: bool) -> int:
    """Caller tensors live during one call: fwd X, Y, W1, W2, b1, b2;
    bwd X, dY, dX, W1, W2, b1, b2 + fp32 dW1, dW2, db1, db2."""
    if not backward:
        return (2 * T * h + 2 * h * f + f + h) * e
    return (3 * T * h + 2 * h * f + f + h) * e + (2 * h * f + f + h) * 4
