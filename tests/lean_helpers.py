"""Test-side glue between the library's exported operator blocks (`dmrg_env_export_block`) and the oracle's
`dmrg.Block` containers, for the output-block-sampled parity tests at BASELINE configs 3-4.

Only marshalling: names, index orders and sector-label conventions of the two sides (include/dmrg_b200.h on one
side, oracle/dmrg.py on the other).  All arithmetic that produces an expected value is done by `oracle/`.
"""
import numpy as np

from oracle import dmrg as odmrg
from oracle.blockops import BlockOp

# library kinds (dmrg_env_export) and the change of (n_up, n_dn) of each class
KINDS = {"H": 0, "CU": 1, "CD": 2, "AUU": 3, "AUD": 4, "ADD": 5, "BUU": 6, "BUD": 7, "BDD": 8, "SU": 9, "SD": 10}
DQ = {"H": (0, 0), "CU": (1, 0), "CD": (0, 1), "AUU": (2, 0), "AUD": (1, 1), "ADD": (0, 2), "BUU": (0, 0), "BUD": (1, -1),
      "BDD": (0, 0), "SU": (-1, 0), "SD": (0, -1)}


def pad8(x):
    return (x + 7) & ~7


def tile_shapes(dL, dR):
    """Tile shapes (row class, col class) in {32, 64, 128}^2 the planner cuts an output block into (csrc/plan.cu
    split_dim, on the dims padded to 8): used to choose sample blocks that span every kernel instance."""
    def split(n):
        out, pos = [], 0
        while pos < n:
            rem = n - pos
            if rem > 96:
                out.append(128); pos += 128
            elif rem > 32:
                out.append(64); pos += 64
            else:
                out.append(32); pos += 32
        return out
    return {(r, c) for r in split(pad8(dL)) for c in split(pad8(dR))}


def choose_blocks(pb, n_random, seed, max_elems=None):
    """Indices of psi blocks: for each of the nine tile shapes the smallest block whose tiling contains it, the
    largest block (the heaviest output: split-K, touched by every workspace chunk), and n_random others."""
    size = [b[4] * b[5] for b in pb]
    chosen = []
    for r in (32, 64, 128):
        for c in (32, 64, 128):
            cand = [i for i, b in enumerate(pb) if (r, c) in tile_shapes(b[4], b[5]) and min(b[4], b[5]) > 8]
            if cand:
                chosen.append(min(cand, key=lambda i: size[i]))
    chosen.append(int(np.argmax(size)))
    rng = np.random.default_rng(seed)
    pool = [i for i in range(len(pb)) if max_elems is None or size[i] <= max_elems]
    chosen += rng.choice(pool, size=min(n_random, len(pool)), replace=False).tolist()
    return sorted(set(int(i) for i in chosen))


class ExportedSide:
    """Reads sector blocks of the carried operators of one block of the library (side 0/1 current, 2/3 cached
    predecessor) and hands them out under the oracle's names, keyed by the block's own electron content."""

    def __init__(self, d, side, orbs, sectors_content, N):
        self.d, self.side = d, side
        self.left = side in (0, 2)
        self.orbs = list(orbs)
        self.sectors = dict(sectors_content)
        self.N = N
        self.bytes = 0

    def _label(self, q):          # content -> label convention of the export call
        return q if self.left else (self.N[0] - q[0], self.N[1] - q[1])

    def _fetch(self, kind, q_in):
        a = self.d.env_export_block(self.side, KINDS[kind], self._label(q_in))
        if a is not None:
            self.bytes += a.nbytes
        return a

    def block(self, keep_q, L, want=("H", "C", "A", "B", "S"), s_orbs=None):
        """dmrg.Block holding, for every carried operator, the sector blocks whose out or in sector is in keep_q."""
        lo = self.orbs[0] if self.orbs else 0
        n = len(self.orbs)
        blk = odmrg.Block(self.orbs, self.sectors)
        ops = blk.ops

        def pairs_in(kind):        # (q_out, q_in) pairs of the class that touch keep_q
            du, dd = DQ[kind]
            out = set()
            for q in keep_q:
                out.add(((q[0] + du, q[1] + dd), q))           # in = q
                out.add((q, (q[0] - du, q[1] - dd)))           # out = q
            return [(qo, qi) for qo, qi in out if qo in self.sectors and qi in self.sectors]

        def fill(kind, names, transform=None):
            """names[idx] = (oracle name, sign, transpose) or None"""
            for qo, qi in pairs_in(kind):
                a = self._fetch(kind, qi)
                if a is None:
                    continue
                assert a.shape[1:] == (self.sectors[qo], self.sectors[qi])
                for idx, spec in enumerate(names):
                    if spec is None:
                        continue
                    for name, sign, tr in spec:
                        op = ops.setdefault(name, BlockOp())
                        m = a[idx] if sign > 0 else -a[idx]
                        if tr:
                            op[(qi, qo)] = m.T
                        else:
                            op[(qo, qi)] = m

        if "H" in want:
            ops["H"] = BlockOp()
            fill("H", [[("H", 1, False)]])
        if "C" in want:
            for s, kind in ((0, "CU"), (1, "CD")):
                for a in range(n):
                    ops[("C", 2 * (lo + a) + s)] = BlockOp()
                fill(kind, [[(("C", 2 * (lo + a) + s), 1, False)] for a in range(n)])
        if "A" in want:
            so = [2 * i + s for i in self.orbs for s in (0, 1)]
            for x, p in enumerate(so):
                for q in so[x + 1:]:
                    ops[("A", p, q)] = BlockOp()
            tri = [(a, b) for a in range(n) for b in range(a + 1, n)]
            fill("AUU", [[(("A", 2 * (lo + a), 2 * (lo + b)), 1, False)] for a, b in tri])
            fill("ADD", [[(("A", 2 * (lo + a) + 1, 2 * (lo + b) + 1), 1, False)] for a, b in tri])
            # a+_iu a+_jd: oracle name ('A', 2i, 2j+1) for i <= j, else -('A', 2j+1, 2i)
            fill("AUD", [[(("A", 2 * (lo + a), 2 * (lo + b) + 1), 1, False)] if a <= b else
                         [(("A", 2 * (lo + b) + 1, 2 * (lo + a)), -1, False)] for a in range(n) for b in range(n)])
        if "B" in want:
            so = [2 * i + s for i in self.orbs for s in (0, 1)]
            for p in so:
                for q in so:
                    ops[("B", p, q)] = BlockOp()
            sq = [(a, b) for a in range(n) for b in range(n)]
            fill("BUU", [[(("B", 2 * (lo + a), 2 * (lo + b)), 1, False)] for a, b in sq])
            fill("BDD", [[(("B", 2 * (lo + a) + 1, 2 * (lo + b) + 1), 1, False)] for a, b in sq])
            # a+_iu a_jd = ('B', 2i, 2j+1);  its transpose a+_jd a_iu = ('B', 2j+1, 2i)
            fill("BUD", [[(("B", 2 * (lo + a), 2 * (lo + b) + 1), 1, False), (("B", 2 * (lo + b) + 1, 2 * (lo + a)), 1, True)]
                         for a, b in sq])
        if "S" in want:
            ext = [x for x in range(L) if x not in self.orbs]
            for s, kind in ((0, "SU"), (1, "SD")):
                for x in ext:
                    ops[("S", 2 * x + s)] = BlockOp()
                fill(kind, [[(("S", 2 * x + s), 1, False)] if (s_orbs is None or x in s_orbs) else None for x in ext])
        return blk


def rel_block_errors(got, ref):
    """(rel-L2, max-abs / max-abs(ref)) of one block."""
    nr = np.linalg.norm(ref)
    return np.linalg.norm(got - ref) / nr, np.abs(got - ref).max() / np.abs(ref).max()
