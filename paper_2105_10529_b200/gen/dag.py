"""Tiny symbolic real-arithmetic DAG used by the build-time amplitude generator.

The matrix-element code of PAPER.md:47,67 (wavefunctions -> vertices/propagators -> amplitudes ->
helicity/colour aggregation) is written once in Python on top of `R` (real) and `Cx` (complex)
values; every operation appends a node to a hash-consed DAG with
  * constant folding and structural-zero propagation (the incoming gluons' polarisation vectors
    are mostly zeros: nothing is emitted for them),
  * signs carried on references (a negation never costs an instruction: it folds into DFMA/DADD),
  * common-subexpression elimination (helicity recycling of shared sub-currents is automatic),
  * sums of products built directly as FMA chains (high DFMA fraction on the FP64 pipe),
  * automatic loop-invariant hoisting: nodes that do not depend on a loop symbol are emitted
    before the helicity loop.
The DAG can be (a) emitted as straight-line CUDA device code with exact add/mul/fma counts and
(b) evaluated numerically with NumPy (host-side self-test of the generator).
"""
import numpy as np


class R:
    """A signed reference to a DAG node, or a constant (node is None)."""
    __slots__ = ("g", "n", "s", "c")

    def __init__(self, g, n=None, s=1, c=0.0):
        self.g, self.n, self.s, self.c = g, n, s, c

    # ---- helpers -------------------------------------------------------------------------------
    def is_const(self):
        return self.n is None

    def is_zero(self):
        return self.n is None and self.c == 0.0

    def __neg__(self):
        return R(self.g, None, 1, -self.c) if self.n is None else R(self.g, self.n, -self.s)

    def _lift(self, o):
        return o if isinstance(o, R) else R(self.g, None, 1, float(o))

    def __add__(self, o):
        return self.g.add(self, self._lift(o))

    __radd__ = __add__

    def __sub__(self, o):
        return self.g.add(self, -self._lift(o))

    def __rsub__(self, o):
        return self.g.add(self._lift(o), -self)

    def __mul__(self, o):
        if isinstance(o, Cx):
            return o * self
        return self.g.mul(self, self._lift(o))

    __rmul__ = __mul__


class Dag:
    def __init__(self):
        self.nodes = []          # (op, a, b, c) with operands = node ids or ('k', const)
        self.dep = []            # depends on a loop symbol
        self.cse = {}
        self.names = {}          # node id -> input / symbol name

    # ---- node creation -------------------------------------------------------------------------
    def _new(self, key, dep):
        i = self.cse.get(key)
        if i is None:
            i = len(self.nodes)
            self.nodes.append(key)
            self.dep.append(dep)
            self.cse[key] = i
        return i

    def const(self, v):
        return R(self, None, 1, float(v))

    def inp(self, name):
        i = self._new(("in", name, None, None), False)
        self.names[i] = name
        return R(self, i)

    def sym(self, name):
        i = self._new(("sym", name, None, None), True)
        self.names[i] = name
        return R(self, i)

    def xl(self, slot, k, rnd=0):
        """value of exchange slot `slot` as stored by the lane `k` places on (gen/lanes.py: one event over several lanes);
        a body node without operands, emitted as a load.  rnd tells apart the uses of a slot that is written more than once."""
        return R(self, self._new(("xl", slot, k, rnd), True))

    def _d(self, *rs):
        return any(r.n is not None and self.dep[r.n] for r in rs)

    def mul(self, a, b):
        if a.is_zero() or b.is_zero():
            return self.const(0.0)
        if a.is_const() and b.is_const():
            return self.const(a.c * b.c)
        if b.is_const():
            a, b = b, a
        if a.is_const():                      # constant * node
            if a.c == 1.0:
                return b
            if a.c == -1.0:
                return -b
            s = b.s * (1 if a.c > 0 else -1)
            return R(self, self._new(("mulk", b.n, abs(a.c), None), self.dep[b.n]), s)
        x, y = (a.n, b.n) if a.n <= b.n else (b.n, a.n)
        return R(self, self._new(("mul", x, y, None), self._d(a, b)), a.s * b.s)

    def add(self, a, b):
        if a.is_zero():
            return b
        if b.is_zero():
            return a
        if a.is_const() and b.is_const():
            return self.const(a.c + b.c)
        if a.is_const():
            a, b = b, a
        if b.is_const():                      # node + constant
            # s*(x) + k  =  s * (x + s*k)
            return R(self, self._new(("addk", a.n, a.s * b.c, None), self.dep[a.n]), a.s)
        if a.n == b.n:
            return self.mul(self.const(2.0), a) if a.s == b.s else self.const(0.0)
        if a.s == b.s:
            x, y = (a.n, b.n) if a.n <= b.n else (b.n, a.n)
            return R(self, self._new(("add", x, y, None), self._d(a, b)), a.s)
        # a - b (signs differ): canonical sub(x, y) with x < y
        pos, neg = (a, b) if a.s > 0 else (b, a)
        if pos.n < neg.n:
            return R(self, self._new(("sub", pos.n, neg.n, None), self._d(a, b)), 1)
        return R(self, self._new(("sub", neg.n, pos.n, None), self._d(a, b)), -1)

    def fma(self, a, b, c):
        """a*b + c as one node (falls back to mul/add when an operand is constant or zero)."""
        if a.is_zero() or b.is_zero():
            return c
        if c.is_zero():
            return self.mul(a, b)
        if a.is_const() and b.is_const():
            return self.add(self.const(a.c * b.c), c)
        if c.is_const():
            return self.add(self.mul(a, b), c)
        if b.is_const():
            a, b = b, a
        if a.is_const():
            if abs(a.c) == 1.0:
                return self.add(self.mul(a, b), c)
            sp = b.s * (1 if a.c > 0 else -1)
            key_ab = ("k", abs(a.c), b.n)
        else:
            sp = a.s * b.s
            x, y = (a.n, b.n) if a.n <= b.n else (b.n, a.n)
            key_ab = ("n", x, y)
        dep = self._d(a, b, c)
        if sp == c.s:
            return R(self, self._new(("fma", key_ab, c.n, None), dep), sp)
        return R(self, self._new(("fms", key_ab, c.n, None), dep), sp)     # sp*(ab - c)

    def rcp(self, a):
        if a.is_const():
            return self.const(1.0 / a.c)
        return R(self, self._new(("rcp", a.n, None, None), self.dep[a.n]), a.s)

    def sop(self, pairs, addend=None):
        """sum of products as one FMA chain: addend + sum a_i*b_i."""
        acc = addend if addend is not None else self.const(0.0)
        live = [(a, b) for a, b in pairs if not (a.is_zero() or b.is_zero())]
        for a, b in live:
            acc = self.fma(a, b, acc)
        return acc

    def plan(self, outputs, max_cost=None, rcp_leaf=False):
        """Split the live nodes into (prologue, body, hoisted).  max_cost None: every loop-invariant
        node is hoisted.  Otherwise only EXPENSIVE invariants (cone with a reciprocal or more than
        max_cost operations) that the body uses are hoisted; cheap ones are recomputed inside the
        loop (and also in the prologue where a hoisted node needs them), because hoisting everything
        keeps more values alive across the loop than the register file holds.  rcp_leaf: a reciprocal is always
        hoisted, but counts as a leaf for the values built on it (they are recomputed when their cone is small)."""
        mark = self.live(outputs)
        ids = [i for i in range(len(self.nodes)) if mark[i]]
        leaf = lambda i: self.nodes[i][0] in ("in", "sym")
        if max_cost is None:
            pro = [i for i in ids if not self.dep[i] and not leaf(i)]
            body = [i for i in ids if self.dep[i] and not leaf(i)]
            return pro, body, set(pro)
        cone = {}
        for i in ids:
            if self.dep[i]:
                continue
            if leaf(i):
                cone[i] = frozenset()
                continue
            c, big = {i}, self.nodes[i][0] == "rcp"
            for o in self._operands(i):
                if cone[o] is None:
                    if rcp_leaf and self.nodes[o][0] == "rcp":
                        continue                    # the reciprocal itself is hoisted; what is built on it may be recomputed
                    big = True
                else:
                    c |= cone[o]
            cone[i] = None if (big or len(c) > max_cost) else frozenset(c)
        body, hoisted = set(), set()
        stack = [i for i in ids if self.dep[i] and not leaf(i)]
        while stack:
            i = stack.pop()
            if i in body:
                continue
            body.add(i)
            for o in self._operands(i):
                if self.dep[o] or leaf(o):
                    continue
                if cone[o] is None:
                    hoisted.add(o)
                else:
                    stack.append(o)
        pro, stack = set(), list(hoisted)
        while stack:
            i = stack.pop()
            if i in pro or leaf(i):
                continue
            pro.add(i)
            stack.extend(self._operands(i))
        return sorted(pro), sorted(body), hoisted

    # ---- emission order ------------------------------------------------------------------------
    def _factors(self, i):
        """node ids of the multiplicands of a mul/fma node (the operands that can sit in a reuse slot)"""
        op, a, b, c = self.nodes[i]
        if op == "mul":
            return (a, b)
        if op == "mulk":
            return (a,)
        if op in ("fma", "fms"):
            return (a[2],) if a[0] == "k" else (a[1], a[2])
        return ()

    def schedule(self, ids, window=48, distance=3):
        """Reorder `ids` (a topologically ordered list) for the FP64 pipe of sm_100: a DFMA whose three
        64-bit register operands are all fresh takes 3 register-read cycles instead of the pipe's 2
        (profiles/r1_dfma_operands.md: 25 instead of 34 TFLOP/s), one that shares a multiplicand with
        the previous instruction reads it from the operand-reuse cache.  Greedy list scheduling inside
        a sliding window of `window` statements (bounds the extra register pressure): prefer a ready
        statement that (1) does not depend on the last `distance` emitted statements (DFMA latency is
        ~4 issue slots), (2) shares a multiplicand with the previous statement, (3) comes first in
        the original order."""
        if window <= 1:
            return list(ids)
        idset = set(ids)
        pos = {n: k for k, n in enumerate(ids)}
        deps = {n: [o for o in set(self._operands(n)) if o in idset] for n in ids}
        fac = {n: set(self._factors(n)) for n in ids}
        users = {n: [] for n in ids}
        for n in ids:
            for o in deps[n]:
                users[o].append(n)
        waiting = {n: len(deps[n]) for n in ids}
        ready = {n for n in ids if waiting[n] == 0}
        out, done, ptr = [], set(), 0
        while len(out) < len(ids):
            while ids[ptr] in done:
                ptr += 1
            lim = ptr + window
            recent = set(out[-distance:]) if distance > 0 else set()
            prev = fac[out[-1]] if out else set()
            best, bs = None, None
            for n in ready:
                if pos[n] >= lim:
                    continue
                sc = (not any(d in recent for d in deps[n]), bool(fac[n] & prev), -pos[n])
                if bs is None or sc > bs:
                    best, bs = n, sc
            if best is None:                       # nothing ready inside the window: take the first ready one
                best = min(ready, key=lambda n: pos[n])
            ready.discard(best)
            done.add(best)
            out.append(best)
            for u in users[best]:
                waiting[u] -= 1
                if waiting[u] == 0:
                    ready.add(u)
        return out

    # ---- analysis ------------------------------------------------------------------------------
    def _operands(self, i):
        op, a, b, c = self.nodes[i]
        if op in ("in", "sym", "xl"):
            return ()
        if op in ("mulk", "addk", "rcp"):
            return (a,)
        if op in ("mul", "add", "sub"):
            return (a, b)
        if op in ("fma", "fms"):
            return ((a[2],) if a[0] == "k" else (a[1], a[2])) + (b,)
        raise ValueError(op)

    def live(self, outputs):
        mark = [False] * len(self.nodes)
        stack = [r.n for r in outputs if r.n is not None]
        while stack:
            i = stack.pop()
            if mark[i]:
                continue
            mark[i] = True
            stack.extend(self._operands(i))
        return mark

    def counts(self, outputs, dep_only=None):
        """exact add/mul/fma/rcp counts of the live nodes (dep_only: None all, True body, False prologue)"""
        mark = self.live(outputs)
        c = dict(add=0, mul=0, fma=0, rcp=0)
        for i, (op, *_rest) in enumerate(self.nodes):
            if not mark[i] or (dep_only is not None and self.dep[i] != dep_only):
                continue
            if op in ("add", "sub", "addk"):
                c["add"] += 1
            elif op in ("mul", "mulk"):
                c["mul"] += 1
            elif op in ("fma", "fms"):
                c["fma"] += 1
            elif op == "rcp":
                c["rcp"] += 1
        return c

    def count_list(self, ids):
        c = dict(add=0, mul=0, fma=0, rcp=0)
        for i in ids:
            op = self.nodes[i][0]
            if op in ("add", "sub", "addk"):
                c["add"] += 1
            elif op in ("mul", "mulk"):
                c["mul"] += 1
            elif op in ("fma", "fms"):
                c["fma"] += 1
            elif op == "rcp":
                c["rcp"] += 1
        return c

    def emit_list(self, ids, name, prefix, indent="  "):
        """C statements for the given nodes (ascending id = topological order); name(j) gives the C
        identifier of operand j"""
        return ["%sconst T %s%d = %s;" % (indent, prefix, i, self._expr(i, name)) for i in ids]

    # ---- emission ------------------------------------------------------------------------------
    @staticmethod
    def _k(v):
        return "T(%r)" % float(v)          # the emitted code is templated on the real type T

    def _expr(self, i, nm):
        op, a, b, c = self.nodes[i]
        if op == "mul":
            return "%s * %s" % (nm(a), nm(b))
        if op == "mulk":
            return "%s * %s" % (nm(a), self._k(b))
        if op == "add":
            return "%s + %s" % (nm(a), nm(b))
        if op == "sub":
            return "%s - %s" % (nm(a), nm(b))
        if op == "addk":
            return "%s + %s" % (nm(a), self._k(b))
        if op == "rcp":
            return "T(1.0) / %s" % nm(a)
        if op == "xl":
            return "MF_XL(%d, %d)" % (a, b)
        if op in ("fma", "fms"):
            x, y = (self._k(a[1]), nm(a[2])) if a[0] == "k" else (nm(a[1]), nm(a[2]))
            return "fma(%s, %s, %s%s)" % (x, y, "-" if op == "fms" else "", nm(b))
        raise ValueError(op)

    def emit(self, outputs, dep, prefix="v", indent="  "):
        """C statements for the live nodes with self.dep == dep, in creation (= topological) order."""
        mark = self.live(outputs)
        nm = lambda j: self.names.get(j, "%s%d" % (prefix, j))
        lines = []
        for i, (op, *_r) in enumerate(self.nodes):
            if not mark[i] or self.dep[i] != dep or op in ("in", "sym"):
                continue
            lines.append("%sconst T %s%d = %s;" % (indent, prefix, i, self._expr(i, nm)))
        return lines

    def ref(self, r, prefix="v"):
        """C expression for a signed reference."""
        if r.n is None:
            return self._k(r.c)
        name = self.names.get(r.n, "%s%d" % (prefix, r.n))
        return name if r.s > 0 else "-" + name

    # ---- numeric evaluation (generator self-test) ----------------------------------------------
    def evaluate(self, outputs, values):
        """values: dict name -> float or ndarray for every input and symbol.  Returns list of values."""
        mark = self.live(outputs)
        val = [None] * len(self.nodes)
        for i, (op, a, b, c) in enumerate(self.nodes):
            if not mark[i]:
                continue
            if op in ("in", "sym"):
                val[i] = np.asarray(values[a], dtype=np.float64)
            elif op == "xl":
                val[i] = np.asarray(values[("xl", a, b, c)], dtype=np.float64)
            elif op == "mul":
                val[i] = val[a] * val[b]
            elif op == "mulk":
                val[i] = val[a] * b
            elif op == "add":
                val[i] = val[a] + val[b]
            elif op == "sub":
                val[i] = val[a] - val[b]
            elif op == "addk":
                val[i] = val[a] + b
            elif op == "rcp":
                val[i] = 1.0 / val[a]
            elif op in ("fma", "fms"):
                p = (a[1] * val[a[2]]) if a[0] == "k" else (val[a[1]] * val[a[2]])
                val[i] = p + val[b] if op == "fma" else p - val[b]
        out = []
        for r in outputs:
            out.append(np.float64(r.c) if r.n is None else r.s * val[r.n])
        return out


class Cx:
    """Complex value over the DAG (re, im are R)."""
    __slots__ = ("re", "im")

    def __init__(self, re, im):
        self.re, self.im = re, im

    @property
    def g(self):
        return self.re.g

    def conj(self):
        return Cx(self.re, -self.im)

    def __neg__(self):
        return Cx(-self.re, -self.im)

    def __add__(self, o):
        if isinstance(o, Cx):
            return Cx(self.re + o.re, self.im + o.im)
        return Cx(self.re + o, self.im)

    __radd__ = __add__

    def __sub__(self, o):
        if isinstance(o, Cx):
            return Cx(self.re - o.re, self.im - o.im)
        return Cx(self.re - o, self.im)

    def __mul__(self, o):
        g = self.g
        if isinstance(o, Cx):
            return Cx(g.sop([(self.re, o.re), (-self.im, o.im)]), g.sop([(self.re, o.im), (self.im, o.re)]))
        o = self.re._lift(o)
        return Cx(self.re * o, self.im * o)

    __rmul__ = __mul__

    def times_i(self):
        return Cx(-self.im, self.re)


def csum_prod(g, pairs, addend=None):
    """addend + sum_i a_i * b_i for complex a_i, b_i as two FMA chains."""
    re_terms, im_terms = [], []
    for a, b in pairs:
        re_terms += [(a.re, b.re), (-a.im, b.im)]
        im_terms += [(a.re, b.im), (a.im, b.re)]
    return Cx(g.sop(re_terms, None if addend is None else addend.re),
              g.sop(im_terms, None if addend is None else addend.im))
