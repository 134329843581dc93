"""ORACLE (test infrastructure, not product code): the EAGLE draft side on the CPU.

What the paper fixes: PAPER.md:92 (section 3.1) "EAGLE ... a lightweight draft model that consumes target-model hidden
states"; PAPER.md:102 a ~250M drafter beside the ~10B student; PAPER.md:359-361 (App. E) the drafter is FP8 too, greedy
drafting = "a single candidate chain", tree drafting = "a tree of candidate continuations ... verified in a single forward
pass of the target model via tree attention".  The drafter's architecture is not described in the paper; it is taken from
the EAGLE paper it cites (feature-level autoregression), restated here (DESIGN.md R-drafter):

  * feature f_p = the target's residual stream after its last decoder layer at position p (what the final RMSNorm + LM head
    read);
  * the drafter predicts the feature of position p from the TOKEN at position p and the feature of position p-1:
        x_p = [ embed(token_p) ; f_{p-1} ]   (2H, fp32)  ->  Q8  ->  FC (H x 2H, E4M3 W8A8, no bias)  ->  h0_p (H)
        f^_p = DecoderLayer(h0)_p     one decoder layer of the target's shape with its OWN KV cache, tree attention over the
                                      drafter's cached context + the node's ancestors, positions = L + depth
        logits_p = target's final RMSNorm + Q8 + LM head applied to f^_p      (the LM head is shared with the target)
    ~ one 8B-shape layer (218M) + FC (33.5M) = 252M parameters: the paper's "250M";
  * committed positions use TRUE target features (after a verify step the drafter re-runs the accepted tokens with the
    target's features: `extend`); draft nodes use the drafter's own predicted feature of their parent;
  * tree expansion over a static topology (workloads.tree_parents): the child of rank r of a node is the token with the
    (r+1)-th largest logit at that node (ties: lower id first); a chain is the rank-0 path.
Only tests/, smoke() and bench.py's cpu legs may import this; it shares no code with paper_2606_18502_b200/.
"""
import numpy as np

from . import verify_oracle as vo

F32 = np.float32


def child_ranks(parents):
    """rank[i] = position of node i among its parent's children in index order (root: 0)."""
    seen, rank = {}, np.zeros(len(parents), dtype=np.int64)
    for i in range(1, len(parents)):
        p = int(parents[i])
        rank[i] = seen.get(p, 0)
        seen[p] = rank[i] + 1
    return rank


def top_k_tokens(logits_row, k):
    """the k tokens with the largest logits, largest first; ties -> lower token id first"""
    order = np.lexsort((np.arange(len(logits_row)), -logits_row.astype(np.float64)))
    return order[:k].astype(np.int32)


class DraftModel:
    """FC + one decoder layer (an OracleModel of one layer) + the target's embedding / final norm / LM head."""

    def __init__(self, target, shape):
        self.target = target
        self.layer = vo.OracleModel(_one_layer(shape), accum=target.accum)
        self.layer.static = target.static          # FP8 KV of the drafter cache would read ("k_cache", 0) of ITS OWN calibration
        self.fc = None                             # (codes [H, 2H], scales [H])
        self.hidden = shape.hidden

    def set_weight(self, kind, bf16_bits):
        if kind == "d_fc":
            self.fc = vo.quantize_weight(bf16_bits)
        else:
            self.layer.set_weight(kind, 0, bf16_bits)


class _Shape:
    pass


def _one_layer(shape):
    s = _Shape()
    for f in ("hidden", "n_q_heads", "n_kv_heads", "head_dim", "ffn", "vocab", "rms_eps", "rope_theta"):
        setattr(s, f, getattr(shape, f))
    s.n_layers = 1
    return s


def draft_forward(dm, dcache, seq, tokens, feats, parents):
    """One drafter pass over the nodes `tokens` (tree given by parents, node 0 at position L = dcache.ctx_len[seq]) whose
    predecessor features are feats [T, H] (fp32).  Writes the drafter's K/V of node i at slot L+i.
    -> (f_hat [T, H], logits [T, V])."""
    x = np.concatenate([vo.embed(dm.target, tokens), np.asarray(feats, dtype=F32)], axis=1)      # [T, 2H]
    xq, sx = vo.quantize_rows(x)
    h0 = vo.linear(xq, sx, dm.fc[0], dm.fc[1], accum=dm.layer.accum)
    L = dcache.ctx_len[seq]
    f_hat = vo.layer_forward(dm.layer, 0, h0, dcache, seq, L, parents)
    return f_hat, vo.lm_head(dm.target, f_hat)


def draft_extend(dm, dcache, seq, tokens, feats):
    """Commit accepted tokens into the drafter's cache with the TARGET's true predecessor features (a chain, every node kept).
    -> (f_hat of the last token, its logits)"""
    par = np.arange(-1, len(tokens) - 1)
    f_hat, logits = draft_forward(dm, dcache, seq, np.asarray(tokens), feats, par)
    dcache.ctx_len[seq] += len(tokens)
    return f_hat[-1], logits[-1]


def expand_tree(dm, dcache, seq, root_token, root_feat, parents):
    """Level-by-level expansion of the static topology: -> (tokens [T], f_hat [T, H]).  Node 0 is the root (the last
    emitted token, predecessor feature root_feat = the target's feature at the node that predicted it); a node of depth d
    gets its token from its parent's logits (rank-th largest) and its predecessor feature from its parent's f_hat.
    Levels are run as growing prefixes of the node list (nodes are ordered by depth): rows are independent given their
    ancestors' K/V, so recomputing the earlier levels changes nothing."""
    parents = np.asarray(parents)
    T = len(parents)
    depth = vo.node_depths(parents)
    rank = child_ranks(parents)
    tokens = np.zeros(T, dtype=np.int32)
    feats = np.zeros((T, dm.hidden), dtype=F32)
    tokens[0] = root_token
    feats[0] = root_feat
    f_hat = None
    for d in range(int(depth.max()) + 1):
        n = int(np.count_nonzero(depth <= d))
        f_hat, logits = draft_forward(dm, dcache, seq, tokens[:n], feats[:n], parents[:n])
        for i in range(n, T):
            if depth[i] == d + 1:
                p = int(parents[i])
                k = int(np.count_nonzero(parents == p))
                tokens[i] = top_k_tokens(logits[p], k)[rank[i]]
                feats[i] = f_hat[p]
    return tokens, f_hat


def speculative_generate(target, tcache, dm, dcache, seq, root, root_feat, parents, n_steps):
    """Closed loop: draft a tree -> verify it with the target (greedy acceptance, KV compaction) -> extend the drafter's cache
    with the accepted tokens and the target's features.  -> (emitted tokens, accepted count per step).  The emitted
    sequence equals the target's plain greedy decode whatever the drafter predicts."""
    out, acc = [], []
    for _ in range(n_steps):
        tokens, _ = expand_tree(dm, dcache, seq, root, root_feat, parents)
        r = vo.verify(target, tcache, seq, tokens, parents, commit=True, want_hidden=True)
        path = r["path"]
        feat = r["hidden"][-1]                                   # target features of all tree nodes
        # accepted tokens = root and the accepted drafts; each one's predecessor feature is the TARGET feature of the node before it
        acc_tokens = [int(tokens[n]) for n in path]
        acc_feats = np.stack([root_feat] + [feat[n] for n in path[:-1]])
        draft_extend(dm, dcache, seq, acc_tokens, acc_feats)
        out += r["out_tokens"]
        acc.append(r["accept_len"])
        root, root_feat = r["out_tokens"][-1], feat[path[-1]]
    return out, acc
