"""fp64 ORACLE for the nearest-neighbour (NN) approximation of the N-body sum.

TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as obem_ref.c): imports nothing from paper_2110_09214_b200 and
shares no code with the CUDA path.  numpy for the bookkeeping; the exact pair sums are the pinned Eq (3.8) oracle
(oracle/ref.py eval_field) called as a library step.

PAPER.md:279-285, section 3.2.4: "a nearest neighbour (NN) approximation method ... consists in evaluating the exact
Coulombian field following (3.8) for each of the closest particles to the particle of interest while the field from
the particles further away is approximated by their centre of charges with a barycentric method."  The paper gives
no more than this sentence (and Fig 6 / Table 2 for its accuracy and speed), so the algorithm below is DESIGN.md
reading A19, followed here step by step:

 1. Partition (a k-d tree with equal-count leaves).  Start with one segment holding all N charges in input order.
    Level by level, every segment [a, b) with more than 256 members is (i) sorted, stably, by the coordinate along the
    axis of the largest extent of its members' bounding box (extents compared in fp64, the first axis wins a tie;
    coordinates ordered by the IEEE total order of their fp32 bit patterns, i.e. -0 before +0) and (ii) cut at
    a + 256 ceil(ceil((b - a)/256) / 2): the left child gets the larger half of the leaves, every leaf but the last of
    the whole array gets exactly 256 members.  Segments of <= 256 members are final.
 2. The order after the last level is the "sorted" order.
 3. Leaf l = sorted positions [256 l, 256 (l+1)): axis-aligned bounding box of its members, and two pseudo-particles:
    Q+ = sum of its positive charges at R+ = sum(q r)/Q+ over them, Q- and R- likewise for the negative ones (the
    centre of charge of a same-sign set is a barycentre with positive weights: always inside the box).
 4. Target group g = sorted positions [2048 g, 2048 (g+1)) (8 leaves): bounding box of its members.
 5. A box B is FAR from group g iff  theta^2 * dist2(box_g, B) > diag2(B), with dist2 the squared distance between the
    boxes (sum over axes of max(0, lo_B - hi_g, lo_g - hi_B)^2, added x, y, z in that order) and diag2 the squared
    diagonal of B; fp64 on the fp32 bounds.  Two levels: super-leaf s = leaves [64 s, 64 (s+1)) (its box = the union of
    their boxes, its two pseudo-particles = the centres of charge of all its positive / negative members).  A super-leaf
    that is FAR from g at the stricter parameter theta/2 (measured on config 3: at theta itself the 16384-charge
    super-leaves triple the error, at theta/2 they leave it unchanged) stands for all its leaves; the leaves of every other super-leaf are classified one by one: FAR
    (its own two pseudo-particles) or NEAR (a group is always near its own leaves: dist2 = 0).
 6. Field and potential at target i of group g:  the exact softened pair sum of Eq (3.8) over every member j != i of
    the near leaves, plus the pseudo-particles of the far super-leaves and of the far leaves (same softening, weight 0
    ones skipped).
 7. Results are returned in the input order.
"""
from __future__ import annotations

import numpy as np

LEAF = 256
GROUP = 2048
SUPER = 64          # leaves per super-leaf
SUPER_THETA = 0.5   # a super-leaf is accepted at half the opening parameter of a leaf


def _ordered_key(f32):
    """fp32 -> uint32 whose unsigned order is the IEEE total order of the floats."""
    u = np.ascontiguousarray(f32, dtype=np.float32).view(np.uint32)
    return np.where(u & np.uint32(0x80000000), ~u, u | np.uint32(0x80000000)).astype(np.uint32)


def split_point(a: int, b: int, leaf: int = LEAF) -> int:
    n_leaves = -(-(b - a) // leaf)
    return a + leaf * (-(-n_leaves // 2))


def kd_order(xyzq, leaf: int = LEAF):
    """Steps 1-2.  xyzq [N, 4] float32 -> perm (int64): sorted position -> input index."""
    x = np.asarray(xyzq, dtype=np.float32)
    n = x.shape[0]
    perm = np.arange(n, dtype=np.int64)
    segs = [(0, n)]
    while any(b - a > leaf for a, b in segs):
        nxt = []
        for a, b in segs:
            if b - a <= leaf:
                nxt.append((a, b))
                continue
            p = x[perm[a:b], :3]
            ext = p.max(axis=0).astype(np.float64) - p.min(axis=0).astype(np.float64)
            ax = int(np.argmax(ext))                                    # first axis of the largest extent
            order = np.argsort(_ordered_key(p[:, ax]), kind="stable")
            perm[a:b] = perm[a:b][order]
            m = split_point(a, b, leaf)
            nxt += [(a, m), (m, b)]
        segs = nxt
    return perm


def build(xyzq, leaf: int = LEAF, group: int = GROUP, super_: int = SUPER):
    """Steps 2-4.  Returns a dict: perm, leaf boxes [nL, 2, 3], pseudo-particles [nL, 2, 4] (+ then -), group boxes."""
    assert group % leaf == 0
    x = np.asarray(xyzq, dtype=np.float32)
    n = x.shape[0]
    perm = kd_order(x, leaf)
    s = x[perm].astype(np.float64)
    n_leaf = (n + leaf - 1) // leaf
    n_group = (n + group - 1) // group
    boxes = np.zeros((n_leaf, 2, 3))
    pseudo = np.zeros((n_leaf, 2, 4))
    for l in range(n_leaf):
        m = s[l * leaf:(l + 1) * leaf]
        boxes[l, 0], boxes[l, 1] = m[:, :3].min(axis=0), m[:, :3].max(axis=0)
        for h, sel in enumerate((m[:, 3] > 0, m[:, 3] < 0)):
            q = m[sel, 3]
            if q.size:
                Q = q.sum()
                pseudo[l, h, :3] = (q[:, None] * m[sel, :3]).sum(axis=0) / Q
                pseudo[l, h, 3] = Q
    n_super = (n_leaf + super_ - 1) // super_
    sboxes = np.zeros((n_super, 2, 3))
    spseudo = np.zeros((n_super, 2, 4))
    for k in range(n_super):
        b = boxes[k * super_:(k + 1) * super_]
        sboxes[k, 0], sboxes[k, 1] = b[:, 0].min(axis=0), b[:, 1].max(axis=0)
        m = s[k * super_ * leaf:(k + 1) * super_ * leaf]
        for h, sel in enumerate((m[:, 3] > 0, m[:, 3] < 0)):
            q = m[sel, 3]
            if q.size:
                Q = q.sum()
                spseudo[k, h, :3] = (q[:, None] * m[sel, :3]).sum(axis=0) / Q
                spseudo[k, h, 3] = Q
    gboxes = np.zeros((n_group, 2, 3))
    per = group // leaf
    for g in range(n_group):
        b = boxes[g * per:(g + 1) * per]
        gboxes[g, 0], gboxes[g, 1] = b[:, 0].min(axis=0), b[:, 1].max(axis=0)
    return {"perm": perm, "sorted": s, "leaf_boxes": boxes, "pseudo": pseudo, "group_boxes": gboxes,
            "super_boxes": sboxes, "super_pseudo": spseudo, "leaf": leaf, "group": group, "super": super_}


def _far(boxes, gb, theta: float):
    """The acceptance test of step 5 for an array of boxes [K, 2, 3] against the group box gb [2, 3]."""
    gap = np.maximum(0.0, np.maximum(boxes[:, 0] - gb[1], gb[0] - boxes[:, 1]))
    dist2 = (gap[:, 0] * gap[:, 0] + gap[:, 1] * gap[:, 1]) + gap[:, 2] * gap[:, 2]
    side = boxes[:, 1] - boxes[:, 0]
    diag2 = (side[:, 0] * side[:, 0] + side[:, 1] * side[:, 1]) + side[:, 2] * side[:, 2]
    return (theta * theta) * dist2 > diag2


def classify(tree, g: int, theta: float):
    """Step 5.  Returns (far_super [nS] bool, near_leaf [nL] bool, far_leaf [nL] bool); a leaf of a far super-leaf is
    neither near nor far on its own."""
    gb = tree["group_boxes"][g]
    far_super = _far(tree["super_boxes"], gb, SUPER_THETA * theta)
    n_leaf = tree["leaf_boxes"].shape[0]
    covered = np.repeat(far_super, tree["super"])[:n_leaf]
    leaf_far = _far(tree["leaf_boxes"], gb, theta)
    return far_super, ~covered & ~leaf_far, ~covered & leaf_far


def far_mask(tree, g: int, theta: float):
    """Boolean [nL]: True where leaf l is NOT summed exactly for group g (far on its own or inside a far super-leaf)."""
    return ~classify(tree, g, theta)[1]


def units(tree, theta: float, n: int, block: int = 256):
    """Source blocks x tiles the GPU form runs: per group its near leaves + ceil(2 (far leaves + far super-leaves) / 256)
    blocks of pseudo-particles."""
    total = 0
    for g in range(tree["group_boxes"].shape[0]):
        fs, near, fl = classify(tree, g, theta)
        total += int(near.sum()) + -(-2 * (int(fl.sum()) + int(fs.sum())) // block)
    return total


def nn_field(xyzq, eps_pp: float, theta: float, leaf: int = LEAF, group: int = GROUP, groups=None, ref=None,
             super_: int = SUPER):
    """Steps 1-7.  Returns out [N, 4] float64 = k_e (Ex, Ey, Ez, phi) in input order (rows of groups that were not
    asked for stay NaN), and the tree.  `groups`: iterable of group indices to evaluate (default all).  `ref`: the
    oracle.ref module (passed in so that this file has no import-time dependency on the compiled library)."""
    if ref is None:
        from oracle import ref as _ref
        ref = _ref
    x = np.asarray(xyzq, dtype=np.float32)
    n = x.shape[0]
    out = np.full((n, 4), np.nan)
    if n == 0:
        return out, None
    tree = build(x, leaf, group, super_)
    perm, s32 = tree["perm"], x[tree["perm"]]
    n_leaf = tree["leaf_boxes"].shape[0]
    n_group = tree["group_boxes"].shape[0]
    for g in (range(n_group) if groups is None else groups):
        far_super, near, far_leaf = classify(tree, g, theta)
        t0, t1 = g * group, min((g + 1) * group, n)
        near_ids = np.nonzero(near)[0]
        members = np.concatenate([np.arange(l * leaf, min((l + 1) * leaf, n)) for l in near_ids])
        # exact part: Eq (3.8) over the members of the near leaves, self excluded by index
        pos_in_members = np.full(n, -1, dtype=np.int64)
        pos_in_members[members] = np.arange(members.size)
        self_index = pos_in_members[t0:t1]
        assert (self_index >= 0).all()
        e_near, _ = ref.eval_field(xyzq=s32[members], targets=s32[t0:t1], self_index=self_index, eps_pp=eps_pp,
                                   flags=ref.NBODY)
        # far part: the two pseudo-particles of every far super-leaf and of every far leaf, in fp64
        pp = np.concatenate([tree["super_pseudo"][far_super].reshape(-1, 4), tree["pseudo"][far_leaf].reshape(-1, 4)])
        pp = pp[pp[:, 3] != 0.0]
        e_far = _pair_sum(s32[t0:t1, :3].astype(np.float64), pp, eps_pp)
        out[perm[t0:t1]] = e_near + e_far
    return out, tree


def _pair_sum(targets, sources, eps):
    """k_e sum_j w_j (r - r_j)/(|r - r_j|^2 + eps^2)^(3/2) and k_e sum_j w_j/(...)^(1/2); fp64, sources [M, 4]."""
    ke = 1.0 / (4.0 * np.pi * 8.8541878128e-12)
    out = np.zeros((targets.shape[0], 4))
    for a in range(0, targets.shape[0], 256):
        d = targets[a:a + 256, None, :] - sources[None, :, :3]
        r2 = (d * d).sum(axis=2) + eps * eps
        with np.errstate(divide="ignore"):
            u = np.where(r2 > 0, 1.0 / np.sqrt(r2), 0.0)
        wu = sources[None, :, 3] * u
        out[a:a + 256, 3] = wu.sum(axis=1)
        out[a:a + 256, :3] = ((wu * u * u)[:, :, None] * d).sum(axis=1)
    return ke * out
