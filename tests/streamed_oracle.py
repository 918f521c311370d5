"""Test helper (imports only oracle/): ONE oracle DM iteration streamed over chunks of views, for problems whose
psi does not fit host memory in complex128 (BASELINE.json configs 3 and 4: 32 / 23 GiB).

It calls the oracle's own steps in oracle_iterate's order (readings A3 / A4 of DESIGN.md): step A per view
(oracle_views_update), eq. (6) with the OLD probe and the new psi accumulated range by range
(oracle_object_accumulate / _finish), then eq. (5) with the NEW object (oracle_probe_accumulate / _finish), and the
error row of eq. (7) with the per-view sums added in ascending j.  psi_new is needed twice (object pass, probe pass):
it is recomputed in the second pass, or, when the caller passes a `stash` (put / get of a chunk, e.g. device memory used
as plain storage), kept from the first.  tests/test_oracle_dm.py requires the result to be
bit-identical to OracleDM.iterate on small problems for several chunk sizes.
"""
import numpy as np

import oracle


def _ordered_sum(values):
    s = 0.0
    for v in values:          # ascending j, one double addition each: oracle_iterate's order
        s += float(v)
    return s


def iteration(positions, P, O, psi_of, amp_of, alpha_obj, alpha_probe, beta=1.0, eps=1e-30, chunk=64, on_psi=None,
              stash=None):
    """P complex128 [K][N][N], O complex128 [L][H][W]: the state before the iteration.
    psi_of(j0, j1) -> complex128 [j1-j0][K][L][N][N] (psi before), amp_of(j0, j1) -> float64 [j1-j0][N][N] (sqrt(I)).
    on_psi(j0, j1, psi_new_chunk), if given, sees every chunk of the new psi once (second pass).
    stash, if given: stash.put(j0, j1, complex128 chunk) in the first pass, stash.get(j0, j1) -> the same bits in the second.
    Returns (P_new, O_new, error row [eps_F, eps_psi, eps_P[0..K), eps_O[0..L)])."""
    pos = np.ascontiguousarray(positions, np.int32)
    P = np.ascontiguousarray(P, np.complex128)
    O = np.ascontiguousarray(O, np.complex128)
    J, K, L = pos.shape[0], P.shape[0], O.shape[0]
    ranges = [(j0, min(J, j0 + chunk)) for j0 in range(0, J, chunk)]
    acc = np.zeros((J, 4))
    numO, denO = np.zeros(O.shape, np.complex128), np.zeros(O.shape[1:], np.float64)
    for j0, j1 in ranges:
        psi_new, acc[j0:j1] = oracle.views_update(pos, j0, j1, P, O, psi_of(j0, j1), amp_of(j0, j1), beta, eps)
        oracle.object_accumulate(pos, j0, j1, P, psi_new, numO, denO)
        if stash is not None:
            stash.put(j0, j1, psi_new)
    O_new = oracle.object_finish(numO, denO, O, alpha_obj)
    numP, denP = np.zeros(P.shape, np.complex128), np.zeros(P.shape[1:], np.float64)
    for j0, j1 in ranges:
        if stash is not None:
            psi_new = stash.get(j0, j1)
        else:
            psi_new, _ = oracle.views_update(pos, j0, j1, P, O, psi_of(j0, j1), amp_of(j0, j1), beta, eps)
        oracle.probe_accumulate(pos, j0, j1, O_new, psi_new, numP, denP)
        if on_psi is not None:
            on_psi(j0, j1, psi_new)
    P_new = oracle.probe_finish(numP, denP, P, alpha_probe)
    s = [_ordered_sum(acc[:, i]) for i in range(4)]
    row = [np.sqrt(s[0] / s[1]) if s[1] > 0 else 0.0, np.sqrt(s[2] / s[3]) if s[3] > 0 else 0.0]
    row += [oracle.rel_change(P_new[k], P[k]) for k in range(K)]
    row += [oracle.rel_change(O_new[l], O[l]) for l in range(L)]
    return P_new, O_new, np.array(row)
