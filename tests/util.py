"""Small helpers shared by the tests (no method arithmetic)."""
import numpy as np
import torch

import oracle


def mk_hdr(site, mask, ctx) -> np.ndarray:
    site = np.asarray(site, dtype=np.uint64)
    mask = np.asarray(mask, dtype=np.uint64)
    ctx = np.asarray(ctx, dtype=np.uint64)
    n = max(site.size, mask.size, ctx.size)
    h = np.empty((n, 2), dtype=np.uint64)
    h[:, 0] = site | (mask << np.uint64(32))
    h[:, 1] = ctx
    return h


def oracle_for(policy) -> "oracle.Oracle":
    return oracle.Oracle(policy.kind, policy.tgt_off, policy.tgts, policy.k0, policy.k1, policy.policy_digest)


def sign_and_tamper_with_oracle(st, orc):
    """tag = oracle sign of the push-time values, then the recorded corruption. Returns tag (torch int64)."""
    tag = orc.sign(st.hdr.cpu().numpy(), st.val.cpu().numpy())
    tag_t = torch.from_numpy(tag.view(np.int64)).to(st.val.device)
    st.apply_return_tamper(tag_t)
    return tag_t


def popc(a) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.uint32)
    return np.unpackbits(a.view(np.uint8).reshape(-1, 4), axis=1).sum(1).astype(np.int64)
