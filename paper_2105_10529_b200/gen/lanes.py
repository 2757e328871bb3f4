"""gg -> t t~ g g with ONE EVENT OVER FOUR LANES (BASELINE.json configs[3], the register-pressure case).

One thread per event cannot hold a helicity configuration of this process: 34 ordered gluon currents
(136 doubles), 41 quark-line spinors (328) and 24 x 2 partial amplitudes (96) -- the one-thread code
spilled 6.5-14 KB per thread and waited on the reloads (profiles/r2_ttgg_ncu.md).  Here the 24 colour
orderings (a b c d) of DESIGN.md 5.3 are split by their LAST gluon d (the one next to the antitop):
lane l of a group of four takes the six orderings that end with gluon l.  Every lane runs the SAME
straight-line code on cyclically relabelled gluons (local label i = global gluon (i + l) mod 4, local
0 = the last gluon), so a warp carries 8 events without divergence:

  * the quark line of a lane is the subtree chi(0) -> chi(c 0) -> chi(b c 0) -> a_(a b c 0), walked depth
    first: 4 spinors alive at a time, no spinor is computed twice in the group;
  * the gluon currents are shared: the cyclic group acts on the 6 / 12 / 12 unordered pairs / triples /
    quadruples (ordered, modulo reflection) with 2 / 3 / 4 orbits; each lane computes one representative
    per orbit, stores it in the warp's shared-memory tile and reads the others from the lane k places on:
    "my j(pi + k)" = "lane l+k's j(pi)"  (MF_XL(slot, k));
  * the colour form uses C_{s s'} = c(s^-1 s') (invariant under relabelling): with the partial amplitudes
    exchanged the same way, lane l adds x_l^T C(0) x_l + 2 x_l^T C(1) x_(l+1) + x_l^T C(2) x_(l+2) with
    lane-independent integer blocks C(k); the four lane sums are added by two shuffles after the loop.

Polarisations: linear basis, unit vectors for all four gluons; the 16 polarisation
assignments are a run-time loop, lambda_4 = + fixed (parity), both lambda_3 unrolled.
"""
import itertools
import numpy as np
from .dag import Dag, R, Cx, csum_prod
from .amplitudes import Gen, colour_matrix

NL = 4
SYNC_STATEMENTS = 2048      # statements between the group barriers of the loop body (B200: 8.9 ms per 1e6 events; 1024: 9.25, 256: 9.4; profiles/r2_tuning.md)


def _canon(pi):
    """(canonical form, sign) with j(pi) = sign * j(canonical): reflection identity j(rev) = (-1)^(k-1) j"""
    pi = tuple(pi)
    rev = tuple(reversed(pi))
    if rev < pi:
        return rev, (1 if len(pi) % 2 == 1 else -1)
    return pi, 1


def _shift(pi, k, nl=NL):
    return tuple((x + k) % nl for x in pi)


def orbits(size, nl=NL):
    """orbits of the cyclic relabelling on the ordered currents of `size` gluons modulo reflection:
    {canonical pi: (representative, k, sign)} with j(pi) = sign * [lane l+k's j(representative)]"""
    out, reps = {}, []
    for pi in itertools.permutations(range(nl), size):
        c, _ = _canon(pi)
        if c in out:
            continue
        reps.append(c)
        for k in range(nl):
            c2, s2 = _canon(_shift(c, k, nl))
            out.setdefault(c2, (c, k, s2))
    return out, reps


class GenLanes(Gen):
    """per-lane program of gg -> t t~ g g; inputs are the lane's relabelled quantities"""

    def __init__(self, nl=NL):
        NL = self.nl = nl                      # gluons = lanes per event (4: gg -> tt~gg; 3: gg -> tt~g)
        self.basis, self.ng, self.g = "linear", NL, Dag()
        self.loop_lam4, self.parity, self.loop_legs = False, True, ()
        g = self.g
        self.input_names = []
        inp = self._inp
        self.mt = inp("mt")
        self.p4 = [inp("p4e"), inp("p4x"), inp("p4y"), inp("p4z")]
        self.t_ing = [inp("t_" + n) for n in ("wp", "wm", "c0", "cx", "cy")]
        self.b_ing = [inp("b_" + n) for n in ("wp", "wm", "c0", "cx", "cy")]
        # all-incoming momenta of the lane's gluons (local label i = global gluon (i + lane) mod 4)
        self.K = [[inp("k%d%s" % (i, c)) for c in "exyz"] for i in range(NL)]
        # unit polarisation vector of local gluon i in this trip of the polarisation loop (loop symbols)
        self.pl = [[g.sym("pl%d%s" % (i, c)) for c in "xyz"] for i in range(NL)]
        self._P, self._j, self._sl, self._chi = {}, {}, {}, {}
        self.orb, self.reps = {}, {}
        for size in range(2, NL + 1):
            o, r = orbits(size, NL)
            self.orb.update(o)
            self.reps[size] = r
        self.slot_of = {}                      # representative -> first of its 4 exchange slots
        self.prog = []                         # ("seg", node count) / ("store", slot, R) / ("sync", round of the loads behind it)
        self.n_slots = 0

    # helicity labels play no role in the memo keys: one symbolic configuration
    def _hk(self, legs, hel):
        return ()

    def pol(self, leg, lam=None):
        zero = self.g.const(0.0)
        return [Cx(zero, zero)] + [Cx(c, zero) for c in self.pl[leg]]

    def j(self, pi, hel=None):
        pi = tuple(pi)
        if len(pi) == 1:
            return self.pol(pi[0])
        c, sgn = _canon(pi)
        if c not in self._j:
            rep, k, s2 = self.orb[c]
            assert k != 0 and rep in self.slot_of, "representative currents are computed in their own phase"
            zero = self.g.const(0.0)
            slot = self.slot_of[rep]
            self._j[c] = [Cx(self.g.xl(slot + m, k) * float(s2), zero) for m in range(4)]
        cur = self._j[c]
        return cur if sgn > 0 else [-x for x in cur]

    def _mark(self):
        self.prog.append(("seg", len(self.g.nodes)))

    def _new_slots(self, n):
        s = self.n_slots
        self.n_slots += n
        return s

    def build(self):
        g = self.g
        NL = self.nl
        num, den, perms = colour_matrix(NL)
        index = {p: i for i, p in enumerate(perms)}
        # ---- gluon currents: one representative per orbit, phase by phase ------------------------------
        for size in range(2, NL + 1):
            for rep in self.reps[size]:
                cur = self._bg(rep, None)
                assert all(c.im.is_zero() for c in cur)
                self._j[rep] = cur
                self.slot_of[rep] = self._new_slots(4)
                self._mark()
                for m in range(4):
                    self.prog.append(("store", self.slot_of[rep] + m, cur[m].re))
            self.prog.append(("sync", 0))
        # ---- quark line: the six orderings (a b c 0), depth first ----------------------------------------
        # orderings (.. c 0) that end with the lane's gluon, grouped so that neighbours share their tails
        local = [tuple(reversed(p)) + (0,) for p in itertools.permutations(range(1, NL))]
        local.sort(key=lambda sg: tuple(reversed(sg)))
        nloc = len(local)
        amps = {1: [], -1: []}
        for sg in local:
            a = self.partial_amps(sg, None, 1)
            amps[1].append(a[1])
            amps[-1].append(a[-1])
        self.local = local
        # ---- colour form with exchanged amplitudes ------------------------------------------------------
        # the exchange tile is reused: all lanes are past their last current load (sync), then store, sync
        self._mark()
        self.prog.append(("sync", 0))
        xs = {}
        slot = 0
        for lam3 in (1, -1):
            for part in ("re", "im"):
                xs[(lam3, part)] = [getattr(a, part) for a in amps[lam3]]
                for i, x in enumerate(xs[(lam3, part)]):
                    self.prog.append(("store", slot + i, x))
                slot += nloc
        self.prog.append(("sync", 1))
        self.n_slots = max(self.n_slots, slot)

        def glob(sg, lane):
            return index[_shift(sg, lane, NL)]

        # blocks C(k) between a lane and the lane k places on; C(NL - k) seen from the other lane is the transpose of C(k):
        # the pairs (k, NL - k), k < NL - k, are taken once with weight 2, the self-paired k = NL / 2 with weight 1
        blocks, weight = {}, {}
        for k in range(0, NL // 2 + 1):
            blk = np.array([[num[glob(si, 0)][glob(sj, k)] for sj in local] for si in local])
            for lane in range(1, NL):          # invariance under relabelling: the blocks do not depend on the lane
                assert (blk == np.array([[num[glob(si, lane)][glob(sj, lane + k)] for sj in local] for si in local])).all()
            blocks[k] = blk
            weight[k] = 1.0 if (k == 0 or 2 * k == NL) else 2.0
        total = g.const(0.0)
        slot = 0
        for lam3 in (1, -1):
            for part in ("re", "im"):
                x = xs[(lam3, part)]
                pairs = []
                for i in range(nloc):
                    y = g.sop([(g.const(2.0 * blocks[0][i][t]), x[t]) for t in range(i + 1, nloc)], g.const(float(blocks[0][i][i])) * x[i])
                    for k in range(1, NL // 2 + 1):
                        y = g.sop([(g.const(weight[k] * blocks[k][i][t]), g.xl(slot + t, k, 1)) for t in range(nloc)], y)
                    pairs.append((x[i], y))
                total = g.sop(pairs, total)
                slot += nloc
        self._mark()
        self.out = total
        self.scale = 2.0 / den                 # parity (lambda_4 fixed) / colour denominator; unit polarisation vectors
        self.blocks = blocks
        return total


# ---- numeric evaluation: the four lanes of one event, segment by segment (generator self-test) ---------
def evaluate_event(gen, mom, mt, ferm, glu_units):
    """|M|^2 body summed over the 16 polarisation assignments and the four lanes.
    mom: [6][4] (g g -> t t~ g g, partonic CM frame); ferm(p, m) -> 5 spinor ingredients;
    glu_units(k) -> (eps1, eps2) unit 3-vectors of an outgoing gluon."""
    g = gen.g
    NL = gen.nl
    Kg = [np.array(mom[0]), np.array(mom[1])] + [-np.array(mom[4 + i]) for i in range(NL - 2)]
    e = [(np.array([1.0, 0.0, 0.0]), np.array([0.0, 1.0, 0.0])), (np.array([1.0, 0.0, 0.0]), np.array([0.0, -1.0, 0.0]))] + \
        [glu_units(mom[4 + i]) for i in range(NL - 2)]
    base = {"mt": mt}
    for n, c in zip(("p4e", "p4x", "p4y", "p4z"), mom[3]): base[n] = c
    for n, c in zip(("wp", "wm", "c0", "cx", "cy"), ferm(mom[2], mt)): base["t_" + n] = c
    for n, c in zip(("wp", "wm", "c0", "cx", "cy"), ferm(mom[3], mt)): base["b_" + n] = c
    total = 0.0
    for ih in range(1 << NL):
        vals = []
        for lane in range(NL):
            v = dict(base)
            for i in range(NL):
                gl = (i + lane) % NL
                for n, c in zip("exyz", Kg[gl]): v["k%d%s" % (i, n)] = c
                pol = e[gl][0] if (ih >> gl) & 1 else e[gl][1]
                for n, c in zip("xyz", pol): v["pl%d%s" % (i, n)] = c
            vals.append(v)
        pending = []
        for item in gen.prog:
            if item[0] == "store":
                pending.append((item[1], item[2]))
            elif item[0] == "sync" and pending:      # the stores before this barrier become readable: round item[1]
                res = [g.evaluate([r for _s, r in pending], vals[lane]) for lane in range(NL)]
                for lane in range(NL):
                    for k in range(1, NL):
                        for (s, _r), x in zip(pending, res[(lane + k) % NL]):
                            vals[lane][("xl", s, k, item[1])] = float(x)
                pending = []
        for lane in range(NL):
            total += float(g.evaluate([gen.out], vals[lane])[0])
    return total


# ---- emission -------------------------------------------------------------------------------------------
def emit_lanes(gen, fname, sched_window=48, sched_distance=5, max_hoist_cost=4):
    """CUDA text of the per-lane function
        template <typename T> T fname(const T* E, const T* G, T* X, T* V, int lane4, int xs0, int xs1, int xs2, int xs3)
    E: the event's table in shared memory: [0..14] = mt, p4, top and antitop spinor ingredients (gen.input_names order), then
       the all-incoming momenta of the four GLOBAL gluons [4][4] (the lane reads its relabelled K_i = E[15 + 4 ((i + lane4) & 3)]);
    G: the event's polarisation table [global gluon][eps1, eps2][x, y, z]; X: the warp's exchange tile [slot][32];
    V: the warp's tile of per-lane loop invariants [NV][32]; lane4: lane within the group of four; xs0 = the thread's lane
    in the warp, xs_k = lane in the warp of the group member k places on.
    Nothing but pointers lives in registers across the polarisation loop: the inputs are re-read from E where they are used,
    the expensive loop invariants (cones with a reciprocal or more than max_hoist_cost operations) are computed once, parked
    in V and re-read; cheap ones are recomputed per trip.  (Hoisting everything kept 221 doubles alive across the loop:
    1.8 KB of local-memory spills per thread, profiles/r2_ttgg_ncu.md.)  The loads cannot be hoisted by the compiler: the
    stores to X may alias them.
    Returns this lane's share of sum_pol sum_{s s'} a_s C a_s'^*; the caller adds the four lanes.  Counts are per LANE and
    event (executed, with the loop-invariant prologue once)."""
    g = gen.g
    NL = gen.nl
    stores = [it[2] for it in gen.prog if it[0] == "store"]
    pro_ids, body_ids, hoisted = g.plan([gen.out] + stores, max_hoist_cost)
    body_set = set(body_ids)
    nh = 1 << NL
    pro, body = g.count_list(pro_ids), g.count_list(body_ids)
    tot = {k: pro[k] + nh * (body[k] + (1 if k == "add" else 0)) for k in pro}
    leaf = lambda j: g.nodes[j][0] in ("in", "sym")
    parked = sorted({o for i in body_ids for o in g._operands(i) if o not in body_set and not leaf(o)})
    vslot = {j: n for n, j in enumerate(parked)}
    n_ev = len(gen.input_names) - 4 * NL            # per-event scalars in front of the gluon momenta
    assert gen.input_names[n_ev] == "k0e" and n_ev == 15
    wrap = "& 3" if NL == 4 else "%% %d" % NL
    in_index = {}
    for idx, n in enumerate(gen.input_names):
        in_index[n] = "%d" % idx if idx < n_ev else "ko%d + %d" % ((idx - n_ev) // 4, (idx - n_ev) % 4)
    U = fname.upper()
    L = ["// GENERATED by paper_2105_10529_b200/gen/lanes.py -- do not edit.",
         "// one event over %d lanes; per LANE and event (executed): %d add, %d mul, %d fma, %d rcp  (flops = add + mul + 2 fma = %d)"
         % (NL, tot["add"], tot["mul"], tot["fma"], tot["rcp"], tot["add"] + tot["mul"] + 2 * tot["fma"]),
         "#define %s_NADD %dull" % (U, tot["add"]), "#define %s_NMUL %dull" % (U, tot["mul"]),
         "#define %s_NFMA %dull" % (U, tot["fma"]), "#define %s_NEV %d" % (U, n_ev + 4 * NL),
         "#define %s_SCALE %r" % (U, gen.scale), "#define %s_SLOTS %d" % (U, gen.n_slots), "#define %s_NV %d" % (U, len(parked))]
    L.append("enum { " + ", ".join("%s_EV_%s = %d" % (U, n.upper(), i) for i, n in enumerate(gen.input_names[:n_ev])) + ", %s_EV_K = %d };" % (U, n_ev))
    L.append("#if defined(__CUDACC__) || defined(MF_LANES_HOST_EMULATION)      // device code (warp barriers, shared-memory tile); the CPU test harness runs it on four host threads")
    L.append("#define MF_XL(s, k) X[(s) * 32 + xs##k]")
    L.append("template <typename T>")
    L.append("MF_DEVFN T %s(const T* E, const T* G, T* X, T* V, const int lane4, %s) {" % (fname, ", ".join("const int xs%d" % k for k in range(NL))))
    for i in range(NL):
        L.append("  const int gl%d = (lane4 + %d) %s, ko%d = %d + 4 * gl%d;" % (i, i, wrap, i, n_ev, i))
    L.append("  {      // loop invariants that are worth keeping: computed once, parked in V")
    used_pro = sorted({o for i in pro_ids for o in g._operands(i) if g.nodes[o][0] == "in"})
    for j in used_pro:
        L.append("    const T %s = E[%s];" % (g.names[j], in_index[g.names[j]]))
    pname = lambda j: g.names[j] if leaf(j) else "p%d" % j
    L += g.emit_list(pro_ids, pname, "p", indent="    ")
    for j in parked:
        L.append("    V[%d * 32 + xs0] = p%d;" % (vslot[j], j))
    L.append("  }")
    L.append("  T acc = T(0.0);")
    L.append("#pragma unroll 1")
    L.append("  for (int ih = 0; ih < %d; ++ih) {" % nh)
    for i in range(NL):
        L.append("    const T* gp%d = G + gl%d * 6 + (((ih >> gl%d) & 1) ? 0 : 3);" % (i, i, i))
        L.append("    const T pl%dx = gp%d[0], pl%dy = gp%d[1], pl%dz = gp%d[2];" % (i, i, i, i, i, i))

    def bname(j):
        if g.nodes[j][0] == "in":
            return "E[%s]" % in_index[g.names[j]]
        if leaf(j):
            return g.names[j]
        return "v%d" % j if j in body_set else "V[%d * 32 + xs0]" % vslot[j]

    lo, nstmt = 0, 0
    for it in gen.prog:
        if it[0] == "seg":
            ids = [i for i in body_ids if lo <= i < it[1]]
            lo = it[1]
            if ids:
                ids = g.schedule(ids, sched_window, sched_distance)
                for line in g.emit_list(ids, bname, "v", indent="    "):
                    if nstmt % SYNC_STATEMENTS == 0:      # group barrier: keeps the four warps of a group on the same I-cache lines
                        L.append("    MF_SYNC_POINT(0);")
                    L.append(line)
                    nstmt += 1
        elif it[0] == "store":
            r = it[2]
            L.append("    X[%d * 32 + xs0] = %s;" % (it[1], g._k(r.c) if r.n is None else ("" if r.s > 0 else "-") + bname(r.n)))
        else:
            L.append("    __syncwarp();")
    L.append("    acc += %s;" % (g._k(gen.out.c) if gen.out.n is None else ("" if gen.out.s > 0 else "-") + bname(gen.out.n)))
    L.append("    __syncwarp();      // the tile is rewritten by the next trip")
    L.append("  }")
    L.append("  return acc;")
    L.append("}")
    L.append("#undef MF_XL")
    L.append("#endif")
    return "\n".join(L) + "\n", tot, dict(pro=pro, body=body, parked=len(parked))
