"""Exact SU(3) colour algebra in the colour-flow (fundamental string) basis for the process generator.

The paper keeps colour outside the HEGET functions: qqg amplitudes carry -T^a (Eq. 38), ggg
carries i f^{abc} (Eq. 44), gggg three f f structures (Eq. 49 / C.48),
and MG2CUDA multiplies the colour-basis amplitudes with a precomputed colour matrix.  Here
every structure is rewritten on strings of generators along the (single) quark line,

    i f^{abc} T^c = [T^a, T^b],

so the colour of any subtree is a linear combination of WORDS (tuples of gluon leg numbers, in matrix-product
order from the end of the fermion arrow to its start).  The colour matrix between two words is a trace, reduced
exactly with the Fierz identity  T^a_ij T^a_kl = 1/2 (d_il d_jk - 1/N d_ij d_kl)  in rational arithmetic.

Kinds of colour objects:
  'none'  no colour content (leptons, electroweak bosons made of leptons)            words: ()
  'col'   quark line open towards the parent at its END   (column spinor subtree)      words: tuple of legs
  'row'   quark line open towards the parent at its START (row spinor subtree)
  'adj'   gluon-type object X^a, represented by X = X^a T^a                           words: tuple of legs
  'open'  gluon-type object X^a = (T^w1 .. T^a .. T^wn)_{ki} containing the whole quark line; the position of
          the free adjoint index is the marker MARK inside the word
  'line'  complete quark line (colour singlet towards the parent)

Two quark lines (weak-boson fusion, Eq. 21-22 of the paper): a quark line that is complete and carries no gluon is a
colour singlet delta_{row, col}; it travels along with whatever object its boson attaches to as a PASSENGER
(`Col.extra`, a tuple of (row leg, column leg) pairs), and `Col.ends` remembers the external legs at the two ends of
the object's own line.  An amplitude with passengers has the colour flow  ('Q', (r1, c1), (r2, c2), ...)  and the
colour matrix between two such flows is N^(number of index loops) times the relative Fermi sign of the two
pairings (`flow_sign`).  Gluons on a line that is, or travels with, a passenger are not implemented (the paper's
Eq. 21a, 22a with n > 2).
"""
from fractions import Fraction

MARK = -1
NC = 3


class Col:
    __slots__ = ('kind', 'terms', 'ends', 'extra')

    def __init__(self, kind, terms, ends=(None, None), extra=()):
        self.kind = kind
        self.terms = {w: c for w, c in terms.items() if c != 0}
        self.ends = ends                    # (row leg, column leg) at the ends of this object's quark line
        self.extra = tuple(sorted(extra))   # complete gluon-free quark lines travelling along: (row, col) pairs

    def __repr__(self):
        return 'Col(%s, %r%s)' % (self.kind, self.terms, (', extra=%r' % (self.extra,)) if self.extra else '')

    def scaled(self, s):
        return Col(self.kind, {w: c * s for w, c in self.terms.items()}, self.ends, self.extra)

    def key(self):
        """What two colour objects must share to be proportional (used when currents are merged)."""
        return (self.kind, frozenset(self.terms), self.ends, self.extra)


def _join(*objs):
    """Passengers of a combination of objects."""
    out = ()
    for o in objs:
        if o is not None:
            out += o.extra
    return out


def _acc(d, w, c):
    d[w] = d.get(w, 0) + c


def leaf(kind, leg=None):
    if kind == 'col':
        return Col(kind, {(): 1}, ends=(None, leg))
    if kind == 'row':
        return Col(kind, {(): 1}, ends=(leg, None))
    return Col(kind, {((leg,) if kind == 'adj' else ()): 1})


def _subst(word, repl_words):
    """Replace MARK in `word` by each (word, coeff) of repl_words."""
    i = word.index(MARK)
    return [(word[:i] + r + word[i + 1:], c) for r, c in repl_words]


def f3(x, y):
    """Colour of  i f^{xyz} X^x Y^y  as an object with free index z (used for ggg and, nested, for gggg)."""
    out = {}
    if x.kind == 'adj' and y.kind == 'adj':  # [X, Y]
        for wx, cx in x.terms.items():
            for wy, cy in y.terms.items():
                _acc(out, wx + wy, cx * cy)
                _acc(out, wy + wx, -cx * cy)
        return Col('adj', out, extra=_join(x, y))
    if x.kind == 'open' and y.kind == 'adj':  # i f^{xyz} T^x Y^y = [Y, T^z]
        for wx, cx in x.terms.items():
            for wy, cy in y.terms.items():
                for w, c in _subst(wx, [(wy + (MARK,), 1), ((MARK,) + wy, -1)]):
                    _acc(out, w, c * cx * cy)
        return Col('open', out, x.ends, _join(x, y))
    if x.kind == 'adj' and y.kind == 'open':  # i f^{xyz} X^x T^y = [T^z, X]
        for wx, cx in x.terms.items():
            for wy, cy in y.terms.items():
                for w, c in _subst(wy, [((MARK,) + wx, 1), (wx + (MARK,), -1)]):
                    _acc(out, w, c * cx * cy)
        return Col('open', out, y.ends, _join(x, y))
    raise ValueError('f3: unsupported colour kinds %s, %s' % (x.kind, y.kind))


def contract(x, y):
    """X^a Y^a for one 'open' and one 'adj' object -> complete line."""
    if x.kind == 'adj' and y.kind == 'open':
        x, y = y, x
    if not (x.kind == 'open' and y.kind == 'adj'):
        raise ValueError('contract: unsupported colour kinds %s, %s' % (x.kind, y.kind))
    out = {}
    for wx, cx in x.terms.items():
        for w, c in _subst(wx, list(y.terms.items())):
            _acc(out, w, c * cx)
    return Col('line', out, x.ends, _join(x, y))


def qqg(col, row, glu):
    """Colour of the T^a_{ji} vertex given any two of (column quark, row quark, gluon) -> the third, or all
    three -> complete line."""
    out = {}
    if col is not None and row is not None and glu is not None:
        for wr, cr in row.terms.items():
            for wg, cg in glu.terms.items():
                for wc, cc in col.terms.items():
                    _acc(out, wr + wg + wc, cr * cg * cc)
        return Col('line', out, (row.ends[0], col.ends[1]), _join(col, row, glu))
    if row is None:
        for wg, cg in glu.terms.items():
            for wc, cc in col.terms.items():
                _acc(out, wg + wc, cg * cc)
        return Col('col', out, col.ends, _join(col, glu))
    if col is None:
        for wr, cr in row.terms.items():
            for wg, cg in glu.terms.items():
                _acc(out, wr + wg, cr * cg)
        return Col('row', out, row.ends, _join(row, glu))
    for wr, cr in row.terms.items():
        for wc, cc in col.terms.items():
            _acc(out, wr + (MARK,) + wc, cr * cc)
    return Col('open', out, (row.ends[0], col.ends[1]), _join(col, row))


def _passenger(line):
    """A complete quark line becomes a passenger of another object: only a gluon-free line (a plain delta) can."""
    if set(line.terms) != {()}:
        raise NotImplementedError('gluons on a quark line that travels with another quark line')
    return line.terms[()], (line.ends,) + line.extra


def singlet(children):
    """Colour of a colourless ('1' / delta) vertex.  One quark line may pass through or be completed here; further
    complete gluon-free lines ride along as passengers."""
    cols = [c for c in children if c.kind == 'col']
    rows = [c for c in children if c.kind == 'row']
    lines = [c for c in children if c.kind == 'line']
    if any(c.kind in ('adj', 'open') for c in children):
        raise ValueError('gluon-type object at a colourless vertex')
    scale = 1
    extra = ()
    for c in children:
        if c.kind == 'none':
            scale *= c.terms[()]
            extra += c.extra
    if len(cols) > 1 or len(rows) > 1:
        raise ValueError('two open quark lines of the same kind at one vertex')
    # complete lines beyond the first object become passengers
    own = None
    if cols or rows:
        carried = lines
    else:
        carried = lines[1:]
        own = lines[0] if lines else None
    for ln in carried:
        c, pairs = _passenger(ln)
        scale *= c
        extra += pairs
    if own is not None:
        r = own.scaled(scale)
        return Col('line', r.terms, own.ends, own.extra + extra)
    if not cols and not rows:
        return Col('none', {(): scale}, extra=extra)
    if cols and not rows:
        r = cols[0].scaled(scale)
        return Col('col', r.terms, cols[0].ends, cols[0].extra + extra)
    if rows and not cols:
        r = rows[0].scaled(scale)
        return Col('row', r.terms, rows[0].ends, rows[0].extra + extra)
    out = {}
    for wr, cr in rows[0].terms.items():
        for wc, cc in cols[0].terms.items():
            _acc(out, wr + wc, cr * cc * scale)
    return Col('line', out, (rows[0].ends[0], cols[0].ends[1]), rows[0].extra + cols[0].extra + extra)


def closed_flow(col):
    """Colour of a complete amplitude as {flow: coefficient}: the gluon word of a single quark line, or
    ('Q', (r1, c1), (r2, c2), ...) for several gluon-free lines."""
    if not col.extra:
        return col
    if col.kind not in ('line', 'none'):
        raise ValueError('amplitude with an open colour index')
    pairs = tuple(col.extra)
    if col.kind == 'line':
        if set(col.terms) != {()}:
            raise NotImplementedError('gluons on a quark line next to another quark line')
        pairs += (col.ends,)
    coeff = col.terms[()]
    return Col(col.kind, {('Q',) + tuple(sorted(pairs)): coeff})


def flow_sign(flow):
    """Fermi sign of a pairing of the external quark legs into lines: parity of (r1, c1, r2, c2, ...) against the
    increasing order of the legs."""
    seq = [l for pair in flow[1:] for l in pair]
    sign = 1
    for i in range(len(seq)):
        for j in range(i + 1, len(seq)):
            if seq[i] > seq[j]:
                sign = -sign
    return sign


def _loops(fa, fb):
    """Number of closed index loops of  prod delta_{r c} (flow a)  x  prod delta_{r c} (flow b)."""
    to_row_a = {c: r for r, c in fa[1:]}
    to_col_b = {r: c for r, c in fb[1:]}
    seen, n = set(), 0
    for c0 in to_row_a:
        if c0 in seen:
            continue
        n += 1
        c = c0
        while c not in seen:
            seen.add(c)
            c = to_col_b[to_row_a[c]]
    return n


# ----------------------------------------------------------------------------- traces
def trace_pairs(word):
    """Tr(T^{w1} ... T^{wm}) with every label appearing exactly twice (summed) -> Fraction."""
    return _traces([tuple(word)])


def _traces(cycles):
    # product of traces; find a repeated label, apply Fierz
    for ci, cyc in enumerate(cycles):
        for i, a in enumerate(cyc):
            # partner in the same cycle
            for j in range(i + 1, len(cyc)):
                if cyc[j] == a:
                    x, y = cyc[i + 1:j], cyc[j + 1:] + cyc[:i]
                    rest = cycles[:ci] + cycles[ci + 1:]
                    # Tr(X T^a Y T^a) = 1/2 Tr X Tr Y - 1/(2N) Tr(XY)
                    return (Fraction(1, 2) * _traces(rest + [x, y])
                            - Fraction(1, 2 * NC) * _traces(rest + [x + y]))
            # partner in another cycle
            for cj in range(ci + 1, len(cycles)):
                oth = cycles[cj]
                if a in oth:
                    j = oth.index(a)
                    x = cyc[i + 1:] + cyc[:i]
                    y = oth[j + 1:] + oth[:j]
                    rest = [c for k, c in enumerate(cycles) if k not in (ci, cj)]
                    # Tr(T^a X) Tr(T^a Y) = 1/2 Tr(XY) - 1/(2N) Tr X Tr Y
                    return (Fraction(1, 2) * _traces(rest + [x + y])
                            - Fraction(1, 2 * NC) * _traces(rest + [x, y]))
    val = Fraction(1)
    for cyc in cycles:
        if len(cyc) != 0:
            raise ValueError('unpaired label in trace')
        val *= NC
    return val


def colour_matrix(words):
    """C[w, w'] = sum over all colours of (T^w)_{ki} conj((T^w')_{ki}) = Tr(T^w (T^w')^dagger)."""
    n = len(words)
    if any(w and w[0] == 'Q' for w in words):
        if not all(w and w[0] == 'Q' for w in words):
            raise NotImplementedError('mixed colour-flow types')
        return [[Fraction(NC) ** _loops(words[a], words[b]) * flow_sign(words[a]) * flow_sign(words[b])
                 for b in range(n)] for a in range(n)]
    return [[trace_pairs(tuple(words[a]) + tuple(reversed(words[b]))) for b in range(n)] for a in range(n)]
