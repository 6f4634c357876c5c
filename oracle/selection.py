"""Stop rules, the per-prompt DARTS rule and active-set compaction (oracle; test infrastructure only).

Paper notation -> this code (DESIGN.md notation map): M -> K (keep), M'_i -> Kp_i,
the paper's K (short count) -> S = K - L_long, L -> L_long, M_up -> M_up (default 2K).

Alg. 2 (prose :426-432 and :479; the printed `else` is lost — DESIGN.md R1):
    for each prompt q_i (in parallel):
        if M'_i < M_up:   T_i <- Rollout(q_i, size=M'_i)                      # dual-end, §4.1.2 :140
                          Y_i <- SelectTopShortest(T_i, S) U SelectTopLongest(T_i, L_long)
        else:             Y_i <- Rollout(q_i, size=M'_i, early_stop=M)        # §4.3.1 :222-224
"the top-L longest selection excludes incomplete and invalid trajectories reaching
the system length limit" (:140, :430).  "the generation process is halted
immediately once M valid trajectories are collected, pruning the heavy-tail
computation for the remaining M'_i - M candidates" (:224).

Status codes: ACTIVE 0, VALID 1 (ended by EOS, natural or forced), TRUNC 2 (hit
max_new without EOS: "incomplete and invalid"), PRUNED 3 (stopped by the early-stop
signal).  Length = number of generated tokens including the terminal EOS (R10).
All ties break towards the smaller sample index j (R6).
"""
import numpy as np

from . import ACTIVE, VALID, TRUNC, PRUNED, MODE_AUTO, MODE_DUAL_END, MODE_SHORTEST_EARLY_STOP


def apply_stop(token, length, forced_len, eos_id, max_new):
    """Stop rules in order (R9-R11).  `length` already
    counts this token.  Returns (token written to the trajectory, new status)."""
    if forced_len is not None and forced_len == length:
        return eos_id, VALID                    # forced EOS (BASELINE.json configs)
    if eos_id >= 0 and token == eos_id:
        return token, VALID                     # natural EOS
    if length == max_new:
        return token, TRUNC                     # "reaching the system length limit" :140
    return token, ACTIVE


def group_mode(Kp_i, K, M_up, mode):
    """EARLY (shortest-only + proactive early stop) iff M'_i >= M_up (:432, R2), else DUAL."""
    if mode == MODE_DUAL_END:
        return "DUAL"
    if mode == MODE_SHORTEST_EARLY_STOP:
        return "EARLY"
    return "EARLY" if Kp_i >= M_up else "DUAL"


def select_early(lens, status, K):
    """Shortest-only: "exclusively samples the top-M shortest trajectories" (:222), M *valid*
    ones (:224).  Order by (class, len, j), class VALID < TRUNC < PRUNED (R8); first K."""
    cls = {VALID: 0, TRUNC: 1, PRUNED: 2}
    order = sorted(range(len(lens)), key=lambda j: (cls[int(status[j])], int(lens[j]), j))
    return order[:K]


def select_dual(lens, status, K, L_long):
    """Dual-end (:140): Y_short = S shortest; Y_long = L_long longest among VALID of the rest (R7);
    if fewer than L_long VALID remain, fill with the next rows of the ascending order (R8).
    Emitted as Y_short ascending, then Y_long ascending by (len, j)."""
    n = len(lens)
    S = K - L_long
    asc = sorted(range(n), key=lambda j: (int(lens[j]), j))
    short = asc[:S]
    rest = asc[S:]
    valid_rest = [j for j in rest if int(status[j]) == VALID]
    # L_long largest len among VALID, ties -> smaller j
    longest = sorted(valid_rest, key=lambda j: (-int(lens[j]), j))[:L_long]
    if len(longest) < L_long:
        fill = [j for j in rest if j not in longest][: L_long - len(longest)]
        longest = longest + fill
    longest = sorted(longest, key=lambda j: (int(lens[j]), j))
    return short + longest


def group_rule(lens, status, Kp_i, K, L_long, M_up, mode):
    """Applied to one prompt after every lock-step decode step.
    `status` is modified in place (ACTIVE -> PRUNED on an early stop).
    Returns the K selected sample indices if the group closes at this step, else None."""
    m = group_mode(Kp_i, K, M_up, mode)
    n_active = sum(1 for s in status if int(s) == ACTIVE)
    n_valid = sum(1 for s in status if int(s) == VALID)
    if m == "EARLY" and n_valid >= K and n_active > 0:
        for j in range(len(status)):            # proactive early stop (:224, :479)
            if int(status[j]) == ACTIVE:
                status[j] = PRUNED
        n_active = 0
    if n_active > 0:
        return None
    if m == "EARLY":
        return select_early(lens, status, K)
    return select_dual(lens, status, K, L_long)


def sel_mask(sel):
    """Bitset of the selected sample indices."""
    mask = 0
    for j in sel:
        mask |= 1 << int(j)
    return mask


def compact(rows, status_of_row):
    """Active-set compaction = stable partition keeping ACTIVE rows in order."""
    return [r for r in rows if int(status_of_row[r]) == ACTIVE]


def length_stats(lens):
    """Per-group mean and (population) variance of response length — sigma^2_L(q_i) of
    PAPER.md:175-181, a by-product of the selection reductions (feeds Alg. 1, NEXT row f1)."""
    x = np.asarray(lens, dtype=np.float64)
    return float(np.mean(x)), float(np.mean((x - np.mean(x)) ** 2))
