"""Classification quality of a track-finding result -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md:93-99, Eq. (2) and (3): for the n'-th turn partition of an event with n turns,
    efficiency  eps_n' = C_{n'->n'} / C_n'
    purity      pi_n'  = C_{n'->n'} / sum_{i=1..n} C_{i->n'}
where C_n' is the number of hits from partition n' and C_{i->n'} the number of hits of partition i classified as
partition n'.  The sum of Eq. (3) runs over turn partitions only: noise hits (truth -1) classified into n' are not in
it (they are reported separately as `noise_into`).  A ratio with a zero denominator is reported as -1.
PAPER.md:71: N_c = number of hits found in common by two independent scans (here: labelled >= 0 by both).
Plain Python loops."""
import numpy as np


def classification_quality(labels, truth, n_turns):
    C = [[0] * n_turns for _ in range(n_turns)]          # C[i][j]: truth i classified as j
    c_true = [0] * n_turns
    noise_into = [0] * n_turns
    for lab, tr in zip(labels, truth):
        lab, tr = int(lab), int(tr)
        if 0 <= tr < n_turns:
            c_true[tr] += 1
            if 0 <= lab < n_turns:
                C[tr][lab] += 1
        elif 0 <= lab < n_turns:
            noise_into[lab] += 1
    eff, pur = [], []
    for k in range(n_turns):
        eff.append(C[k][k] / c_true[k] if c_true[k] else -1.0)
        den = sum(C[i][k] for i in range(n_turns))
        pur.append(C[k][k] / den if den else -1.0)
    return dict(confusion=np.array(C, dtype=np.int32), c_true=np.array(c_true, dtype=np.int32),
                noise_into=np.array(noise_into, dtype=np.int32), efficiency=np.array(eff), purity=np.array(pur))


def common_hits(labels_a, labels_b, turn_a=-1, turn_b=-1):
    """hits that scan A labels turn_a and scan B labels turn_b (-1 = any turn >= 0)"""
    n = 0
    for a, b in zip(labels_a, labels_b):
        a, b = int(a), int(b)
        if (a >= 0 if turn_a < 0 else a == turn_a) and (b >= 0 if turn_b < 0 else b == turn_b):
            n += 1
    return n
