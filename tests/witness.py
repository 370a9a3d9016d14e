"""The generator-side witness: which lanes MUST violate, derived only from the stream's recorded
tamper plan and Python sets — a derivation independent of oracle/ and of the CUDA path
(SURVEY.md §8(c) "Generator witness")."""
import numpy as np

from paper_2606_11871_b200 import streams as S


def expected_viol(st: "S.Stream") -> np.ndarray:
    """uint32 [n] violation masks the construction implies (call after apply_return_tamper)."""
    n = st.n
    want = np.zeros(n, dtype=np.uint32)
    hdr = st.hdr.cpu().numpy().view(np.uint64)
    val = st.val.cpu().numpy().view(np.uint64)
    pol = st.policy
    sets = {}

    def site_set(s):
        if s not in sets:
            sets[s] = set(int(x) for x in pol.tgts[pol.tgt_off[s]:pol.tgt_off[s + 1]])
        return sets[s]

    for plan in (st.ret_tamper, st.fwd_tamper):
        if not len(plan):
            continue
        ev = plan.ev.cpu().numpy()
        lane = plan.lane.cpu().numpy()
        what = plan.what.cpu().numpy()
        for e, l, w in zip(ev, lane, what):
            site = int(hdr[e, 0] & np.uint64(0xFFFFFFFF))
            mask = int(hdr[e, 0] >> np.uint64(32))
            kind = int(pol.kind[site])
            if kind == S.PROTECTED_RETURN:
                assert w in (S.T_TAG_XOR, S.T_VAL_XOR)
                want[e] |= np.uint32(1 << int(l))  # a non-zero xor of tag or continuation
            elif kind == S.PROTECTED_FORWARD:
                lanes = [int(l)] if w != S.T_VAL_SET_ALL else [j for j in range(32) if (mask >> j) & 1]
                for j in lanes:
                    if int(val[e, j]) not in site_set(site):
                        want[e] |= np.uint32(1 << j)
            else:
                raise AssertionError("tamper on a non-protected event")
    return want
