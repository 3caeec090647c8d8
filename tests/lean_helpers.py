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


# ---------------------------------------------------------------------------------------------------------------
# SU(2) contexts: reduced operator blocks -> U(1) operator blocks on the CG-expanded basis (oracle/su2.expand_mps)
# ---------------------------------------------------------------------------------------------------------------
SU2_KINDS = {"H": 0, "C": 1, "A0": 2, "A1": 3, "B0": 4, "B1": 5, "S": 6}
SU2_K2 = {"H": 0, "C": 1, "A0": 0, "A1": 2, "B0": 0, "B1": 2, "S": 1}       # doubled rank
SU2_DN = {"H": 0, "C": 1, "A0": 2, "A1": 2, "B0": 0, "B1": 0, "S": -1}      # particle-number change
_R2 = 0.5 ** 0.5


class ExportedSideSU2:
    """Same interface as ExportedSide for an SU(2) context: the carried operators are irreducible tensor operators
    stored by reduced elements, <S'M'|X^k_q|SM> = <S M; k q|S' M'> X_red[S',S] (include/dmrg_b200.h, DESIGN.md §9:
    C_{+1/2} = a+_up, A^1_{+1} = a+_iu a+_ju (i<j), A^0 = (a+_iu a+_jd - a+_id a+_ju)/sqrt2 (i<=j), B^1_{+1} = -a+_iu a_jd,
    B^0 = (a+_iu a_ju + a+_id a_jd)/sqrt2, S~_{+1/2} = -S_{x,dn}).  `block` expands the needed components with the
    oracle's Clebsch-Gordan coefficients into U(1) operator blocks on the basis oracle/su2.expand_mps defines:
    inside the U(1) sector (n_up, n_dn) the multiplets (N, S) with S >= |S_z| follow each other (`layout`)."""

    def __init__(self, d, side, orbs, layout, N_tot):
        """layout: dict U(1) bond label -> (dim, [((N_label, 2S), offset), ...]) of the block's open bond."""
        from oracle import su2 as osu2
        self.cg = osu2.cg
        self.d, self.side = d, side
        self.left = side in (0, 2)
        self.orbs = list(orbs)
        self.N_tot = N_tot
        n2 = N_tot // 2
        self.N = (n2, n2)
        self.layout = {}
        for lab, (dim, lay) in layout.items():
            qc = lab if self.left else (n2 - lab[0], n2 - lab[1])
            self.layout[qc] = (dim, lay)
        self.sectors = {q: v[0] for q, v in self.layout.items()}
        self.bytes = 0
        self._cache = {}

    def _fetch(self, kind, d2S, lab_in):
        key = (kind, d2S, lab_in)
        if key not in self._cache:
            a = self.d.env_export_block(self.side, SU2_KINDS[kind], lab_in, d2S=d2S)
            if a is not None:
                self.bytes += a.nbytes
            self._cache[key] = a
        return self._cache[key]

    def _component(self, kind, q2, qo, qi):
        """(nops, D_out, D_in) array of the component q2 of every operator of `kind` between the U(1) content sectors."""
        k2, dN = SU2_K2[kind], SU2_DN[kind]
        Do, lay_o = self.layout[qo]
        Di, lay_i = self.layout[qi]
        Mi, Mo = qi[0] - qi[1], qo[0] - qo[1]
        assert Mo - Mi == q2 and (qo[0] + qo[1]) - (qi[0] + qi[1]) == dN
        off_o = {lab: off for lab, off in lay_o}
        out = None
        for (Nl, Si), oi in lay_i:
            for d2S in range(-k2, k2 + 1, 2):
                So = Si + d2S
                lab_o = (Nl + dN if self.left else Nl - dN, So)
                if So < 0 or lab_o not in off_o:
                    continue
                c = self.cg(Si, Mi, k2, q2, So, Mo)
                if c == 0.0:
                    continue
                red = self._fetch(kind, d2S, (Nl, Si))
                if red is None:
                    continue
                if out is None:
                    out = np.zeros((red.shape[0], Do, Di))
                oo = off_o[lab_o]
                out[:, oo:oo + red.shape[1], oi:oi + red.shape[2]] += c * red
        return out

    def block(self, keep_q, L, want=("H", "C", "A", "B", "S"), s_orbs=None):
        lo = self.orbs[0] if self.orbs else 0
        n = len(self.orbs)
        blk = odmrg.Block(self.orbs, self.sectors)
        ops = blk.ops
        comp_cache = {}

        def comp(kind, q2, qo, qi):
            key = (kind, q2, qo, qi)
            if key not in comp_cache:
                comp_cache[key] = self._component(kind, q2, qo, qi)
            return comp_cache[key]

        def pairs(du, dd):
            out = set()
            for q in keep_q:
                out.add(((q[0] + du, q[1] + dd), q))
                out.add((q, (q[0] - du, q[1] - dd)))
            return [(qo, qi) for qo, qi in out if qo in self.sectors and qi in self.sectors]

        def put(name, du, dd, comps):
            """comps: list of (kind, q2, idx, coef)"""
            op = ops.setdefault(name, BlockOp())
            for qo, qi in pairs(du, dd):
                m = None
                for kind, q2, idx, coef in comps:
                    a = comp(kind, q2, qo, qi)
                    if a is None:
                        continue
                    m = coef * a[idx] if m is None else m + coef * a[idx]
                if m is not None:
                    op[(qo, qi)] = m

        tri = lambda a, b: a * n - a * (a + 1) // 2 + (b - a - 1)        # a < b
        tri0 = lambda a, b: a * n - a * (a - 1) // 2 + (b - a)           # a <= b
        if "H" in want:
            put("H", 0, 0, [("H", 0, 0, 1.0)])
        if "C" in want:
            for a in range(n):
                put(("C", 2 * (lo + a)), 1, 0, [("C", 1, a, 1.0)])
                put(("C", 2 * (lo + a) + 1), 0, 1, [("C", -1, a, 1.0)])
        if "A" in want:
            for a in range(n):
                for b in range(a, n):
                    i, j = lo + a, lo + b
                    if a < b:
                        put(("A", 2 * i, 2 * j), 2, 0, [("A1", 2, tri(a, b), 1.0)])
                        put(("A", 2 * i + 1, 2 * j + 1), 0, 2, [("A1", -2, tri(a, b), 1.0)])
                        put(("A", 2 * i, 2 * j + 1), 1, 1, [("A1", 0, tri(a, b), _R2), ("A0", 0, tri0(a, b), _R2)])
                        put(("A", 2 * i + 1, 2 * j), 1, 1, [("A1", 0, tri(a, b), _R2), ("A0", 0, tri0(a, b), -_R2)])
                    else:
                        put(("A", 2 * i, 2 * i + 1), 1, 1, [("A0", 0, tri0(a, a), _R2)])
        if "B" in want:
            for a in range(n):
                for b in range(n):
                    i, j, ix = lo + a, lo + b, a * n + b
                    put(("B", 2 * i, 2 * j), 0, 0, [("B1", 0, ix, _R2), ("B0", 0, ix, _R2)])
                    put(("B", 2 * i + 1, 2 * j + 1), 0, 0, [("B1", 0, ix, -_R2), ("B0", 0, ix, _R2)])
                    put(("B", 2 * i, 2 * j + 1), 1, -1, [("B1", 2, ix, -1.0)])
                    put(("B", 2 * i + 1, 2 * j), -1, 1, [("B1", -2, ix, 1.0)])
        if "S" in want:
            ext = [x for x in range(L) if x not in self.orbs]
            for idx, x in enumerate(ext):
                if s_orbs is not None and x not in s_orbs:
                    ops[("S", 2 * x)] = BlockOp(); ops[("S", 2 * x + 1)] = BlockOp()
                    continue
                put(("S", 2 * x), -1, 0, [("S", -1, idx, 1.0)])          # S_{x,up} = S~_{-1/2}
                put(("S", 2 * x + 1), 0, -1, [("S", 1, idx, -1.0)])      # S_{x,dn} = -S~_{+1/2}
        self._cache.clear()
        return blk
