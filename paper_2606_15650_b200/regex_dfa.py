"""Host-side regex -> DFA compiler for the device regex detector ("custom regex
patterns"; readings D17-D18).

    blob = compile_patterns([(type_id, pattern), ...], max_match=80)      # bytes, handed to anon_regex_load

Runs once per pattern set; no step of the scan runs here (the scan itself is csrc/regex.cu).  The patterns are byte
regexes in a restricted syntax: literals, escapes (\\d \\w \\s \\xHH, any other escaped byte is itself), `.` (any byte
but \\n), classes `[a-z0-9_]` / `[^...]`, groups `(...)` / `(?:...)`, alternation `|`, quantifiers `? * + {m} {m,} {m,n}`.
Anchors, look-arounds, back-references and lazy quantifiers are rejected (the word-boundary rule of D18 is applied by the
kernel, not by the automaton).

Construction: pattern -> AST -> Thompson NFA (counted repeats unrolled) -> one subset-construction DFA over the
union of all patterns, on byte equivalence classes, accepting label = lowest pattern index -> Moore minimisation.
State 0 is the dead state, state 1 the start state.

Blob layout (little-endian):
    u32 magic 'ARX1', n_states, n_classes, n_patterns, max_match, reserved[3]
    u8  class_of[256]
    u8  is_word[256]                  (1 for [0-9A-Za-z_], rule D18)
    u8  type_of_pattern[256]          (entries >= n_patterns are 0)
    i16 accept[n_states]              (-1 = not accepting, else pattern index), padded to a multiple of 4 bytes
    u16 trans[n_states * n_classes]   (row = state)
"""
import struct

import numpy as np

MAGIC = 0x31585241          # 'ARX1'
ALL = (1 << 256) - 1
_WORD = sum(1 << c for c in b"0123456789ABCDEFGHIJKLMNOPQRSTUVWXYZabcdefghijklmnopqrstuvwxyz_")
_DIGIT = sum(1 << c for c in b"0123456789")
_SPACE = sum(1 << c for c in b" \t\n\r\f\v")


class _Parser:
    def __init__(self, pat):
        self.p = pat.encode("latin-1") if isinstance(pat, str) else bytes(pat)
        self.i = 0

    def fail(self, msg):
        raise ValueError("regex %r: %s at offset %d" % (self.p, msg, self.i))

    def peek(self):
        return self.p[self.i] if self.i < len(self.p) else None

    def parse(self):
        node = self.alt()
        if self.i != len(self.p):
            self.fail("unbalanced ')'")
        return node

    def alt(self):
        parts = [self.cat()]
        while self.peek() == ord("|"):
            self.i += 1
            parts.append(self.cat())
        return parts[0] if len(parts) == 1 else ("alt", parts)

    def cat(self):
        parts = []
        while self.peek() is not None and self.peek() not in b"|)":
            parts.append(self.rep())
        return ("cat", parts)

    def rep(self):
        node = self.atom()
        while True:
            c = self.peek()
            if c == ord("?"):
                lo, hi = 0, 1
                self.i += 1
            elif c == ord("*"):
                lo, hi = 0, None
                self.i += 1
            elif c == ord("+"):
                lo, hi = 1, None
                self.i += 1
            elif c == ord("{"):
                j = self.p.find(b"}", self.i)
                if j < 0:
                    self.fail("unterminated {")
                body = self.p[self.i + 1:j].decode()
                try:
                    if "," in body:
                        a, b = body.split(",")
                        lo, hi = int(a), (int(b) if b else None)
                    else:
                        lo = hi = int(body)
                except ValueError:
                    self.fail("bad repeat count")
                if hi is not None and hi < lo:
                    self.fail("bad repeat range")
                self.i = j + 1
            else:
                return node
            if self.peek() in (ord("?"), ord("+")):
                self.fail("lazy / possessive quantifiers are not supported")
            node = ("rep", node, lo, hi)

    def escape(self):
        """After a backslash: returns a byte-set mask."""
        c = self.peek()
        if c is None:
            self.fail("dangling backslash")
        self.i += 1
        if c == ord("d"):
            return _DIGIT
        if c == ord("w"):
            return _WORD
        if c == ord("s"):
            return _SPACE
        if c in b"DWS":
            return ALL ^ {ord("D"): _DIGIT, ord("W"): _WORD, ord("S"): _SPACE}[c]
        if c == ord("x"):
            h = self.p[self.i:self.i + 2]
            self.i += 2
            try:
                return 1 << int(h, 16)
            except ValueError:
                self.fail("bad \\x escape")
        if c == ord("n"):
            return 1 << 10
        if c == ord("t"):
            return 1 << 9
        if c == ord("r"):
            return 1 << 13
        if c in b"bBAZz" or chr(c).isdigit():
            self.fail("anchors and back-references are not supported")
        return 1 << c

    def cls(self):
        neg = False
        if self.peek() == ord("^"):
            neg = True
            self.i += 1
        mask, first = 0, True
        while True:
            c = self.peek()
            if c is None:
                self.fail("unterminated [")
            if c == ord("]") and not first:
                self.i += 1
                break
            first = False
            self.i += 1
            if c == ord("\\"):
                m = self.escape()
                if m & (m - 1):                        # a multi-byte class such as \d: no range from it
                    mask |= m
                    continue
                c = m.bit_length() - 1
            if self.peek() == ord("-") and self.i + 1 < len(self.p) and self.p[self.i + 1] != ord("]"):
                self.i += 1
                d = self.peek()
                self.i += 1
                if d == ord("\\"):
                    m = self.escape()
                    if m & (m - 1):
                        self.fail("bad range end")
                    d = m.bit_length() - 1
                if d < c:
                    self.fail("reversed range")
                for b in range(c, d + 1):
                    mask |= 1 << b
            else:
                mask |= 1 << c
        return (ALL ^ mask) if neg else mask

    def atom(self):
        c = self.peek()
        self.i += 1
        if c == ord("("):
            if self.p[self.i:self.i + 2] == b"?:":
                self.i += 2
            elif self.peek() == ord("?"):
                self.fail("look-arounds / flags are not supported")
            node = self.alt()
            if self.peek() != ord(")"):
                self.fail("missing ')'")
            self.i += 1
            return node
        if c == ord("["):
            return ("set", self.cls())
        if c == ord("."):
            return ("set", ALL ^ (1 << 10))
        if c == ord("\\"):
            return ("set", self.escape())
        if c in b"^$":
            self.fail("anchors are not supported")
        if c in b"?*+{":
            self.fail("nothing to repeat")
        return ("set", 1 << c)


class _NFA:
    def __init__(self):
        self.eps = []          # state -> [targets]
        self.edge = []         # state -> (mask, target) or None

    def new(self):
        self.eps.append([])
        self.edge.append(None)
        return len(self.eps) - 1

    def build(self, node):
        """Thompson fragment (start, end) of an AST node."""
        kind = node[0]
        if kind == "set":
            a, b = self.new(), self.new()
            self.edge[a] = (node[1], b)
            return a, b
        if kind == "cat":
            a = b = self.new()
            for part in node[1]:
                s, e = self.build(part)
                self.eps[b].append(s)
                b = e
            return a, b
        if kind == "alt":
            a, b = self.new(), self.new()
            for part in node[1]:
                s, e = self.build(part)
                self.eps[a].append(s)
                self.eps[e].append(b)
            return a, b
        _k, sub, lo, hi = node
        a = b = self.new()
        for _ in range(lo):
            s, e = self.build(sub)
            self.eps[b].append(s)
            b = e
        if hi is None:                                 # star of one more copy
            s, e = self.build(sub)
            out = self.new()
            self.eps[b] += [s, out]
            self.eps[e] += [s, out]
            return a, out
        out = self.new()
        for _ in range(hi - lo):                       # nested optionals: every copy may leave to `out`
            s, e = self.build(sub)
            self.eps[b] += [s, out]
            b = e
        self.eps[b].append(out)
        return a, out


def _closure(nfa, states):
    seen, stack = set(states), list(states)
    while stack:
        for t in nfa.eps[stack.pop()]:
            if t not in seen:
                seen.add(t)
                stack.append(t)
    return frozenset(seen)


def compile_tables(patterns, max_states=60000):
    """patterns: [pattern, ...].  Returns (class_of u8[256], accept i16[n_states], trans u16[n_states, n_classes])."""
    nfa = _NFA()
    start = nfa.new()
    accept_of = {}
    for k, pat in enumerate(patterns):
        s, e = nfa.build(_Parser(pat).parse())
        nfa.eps[start].append(s)
        accept_of[e] = k
    # byte equivalence classes: bytes that no edge mask tells apart
    masks = sorted({ed[0] for ed in nfa.edge if ed is not None})
    sig = {}
    class_of = np.zeros(256, np.uint8)
    reps = []
    for b in range(256):
        key = tuple((m >> b) & 1 for m in masks)
        if key not in sig:
            sig[key] = len(reps)
            reps.append(b)
        class_of[b] = sig[key]
    ncls = len(reps)

    def label(S):
        ks = [accept_of[s] for s in S if s in accept_of]
        return min(ks) if ks else -1

    s0 = _closure(nfa, [start])
    if label(s0) >= 0:
        raise ValueError("pattern %d matches the empty string" % label(s0))
    ids = {frozenset(): 0, s0: 1}
    order = [frozenset(), s0]
    rows = [[0] * ncls]
    todo = [s0]
    while todo:
        S = todo.pop()
        row = []
        for b in reps:
            T = _closure(nfa, [nfa.edge[s][1] for s in S if nfa.edge[s] is not None and (nfa.edge[s][0] >> b) & 1])
            if T not in ids:
                ids[T] = len(order)
                order.append(T)
                todo.append(T)
                if len(order) > max_states:
                    raise ValueError("DFA has more than %d states" % max_states)
            row.append(ids[T])
        while len(rows) <= ids[S]:
            rows.append(None)
        rows[ids[S]] = row
    n = len(order)
    trans = np.asarray([r if r is not None else [0] * ncls for r in rows], np.int64).reshape(n, ncls)
    acc = np.asarray([label(S) for S in order], np.int64)

    # Moore minimisation: refine the partition by accept label until transitions respect it
    block = np.unique(acc, return_inverse=True)[1]
    while True:
        key = np.concatenate([block[:, None], block[trans]], axis=1)
        nb = np.unique(key, axis=0, return_inverse=True)[1].reshape(-1)
        if nb.max() == block.max():
            break
        block = nb
    # renumber: dead block -> 0, start block -> 1, the rest in order of first appearance
    remap = {int(block[0]): 0}
    if int(block[1]) in remap:
        raise ValueError("no pattern can match anything")
    remap[int(block[1])] = 1
    for b in block:
        if int(b) not in remap:
            remap[int(b)] = len(remap)
    m = len(remap)
    t2 = np.zeros((m, ncls), np.uint16)
    a2 = np.full(m, -1, np.int16)
    for s in range(n):
        d = remap[int(block[s])]
        t2[d] = [remap[int(block[t])] for t in trans[s]]
        a2[d] = acc[s]
    assert not t2[0].any() and a2[0] < 0
    return class_of, a2, t2


def compile_patterns(typed_patterns, max_match=80):
    """typed_patterns: [(type_id, pattern), ...] in priority order.  Returns the blob for anon_regex_load."""
    if not 1 <= len(typed_patterns) <= 127:
        raise ValueError("1..127 patterns")
    if not 1 <= max_match <= 255:
        raise ValueError("max_match must be in [1, 255]")
    class_of, accept, trans = compile_tables([p for _t, p in typed_patterns])
    if trans.shape[0] > 65535:
        raise ValueError("too many DFA states for 16-bit transitions")
    types = np.zeros(256, np.uint8)
    for k, (t, _p) in enumerate(typed_patterns):
        if not 0 <= int(t) <= 255:
            raise ValueError("type id out of range")
        types[k] = int(t)
    is_word = np.asarray([(_WORD >> b) & 1 for b in range(256)], np.uint8)
    head = struct.pack("<8I", MAGIC, trans.shape[0], trans.shape[1], len(typed_patterns), max_match, 0, 0, 0)
    acc = accept.astype("<i2").tobytes()
    acc += b"\0" * (-len(acc) % 4)
    return head + class_of.tobytes() + is_word.tobytes() + types.tobytes() + acc + trans.astype("<u2").tobytes()
