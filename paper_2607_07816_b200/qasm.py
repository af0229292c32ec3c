"""OpenQASM 2.0 reader (optional part; Fig. 1: the paper's circuits arrive as
OpenQASM 2.0 text that includes "qelib1.inc" and applies u3 and cz; PAPER.md:57 refers to that gate list).

Host-side text parsing only: the result is a `workloads.Circuit` -- a list of (name, qubits, U) records in the
conventions of `workloads.py` (qubit q = bit q of the key, U row-major with local bit j = qubits[j]; R1, R2,
R16) -- which feeds `engine.SparseSV.apply_circuit`, `engine.fuse_gates` / `reorder_gates` or the CPU oracle alike.
Like `workloads.py` this module holds none of the method's arithmetic.

Supported: the header, `include` (ignored: the qelib1 gates below are built in), any number of `qreg` (qubits are
numbered in declaration order), `creg` / `measure` / `barrier` (ignored: the simulator reads the whole state out),
register broadcast (`h q;`, `cx a, b;` with registers of equal size), and the gates
    U / u3, u2, u1, u0, id, x, y, z, h, s, sdg, t, tdg, rx, ry, rz, cx / CX, cy, cz, ch, swap, ccx, cswap, crz, cu1, cu3, rzz
with parameter expressions over numbers, `pi`, + - * / ^, parentheses and sin cos tan exp ln sqrt.
Not supported (a ValueError names the statement): `gate` / `opaque` definitions, `if`, `reset`.

rz(theta) is diag(e^{-i theta/2}, e^{i theta/2}) (R16); it differs from qelib1's u1(theta) by a global phase,
which no probability depends on.
"""
from __future__ import annotations

import math
import re
from typing import Dict, List, Tuple

import numpy as np

from . import workloads as W

C128 = np.complex128


# ---- parameter expressions: recursive descent, no eval --------------------------------------------
_TOK = re.compile(r"\s*(?:(\d+\.\d*(?:[eE][+-]?\d+)?|\.\d+(?:[eE][+-]?\d+)?|\d+(?:[eE][+-]?\d+)?)|([A-Za-z_]\w*)|(.))")
_FUNCS = {"sin": math.sin, "cos": math.cos, "tan": math.tan, "exp": math.exp, "ln": math.log, "sqrt": math.sqrt}


def eval_expr(text: str) -> float:
    toks: List[Tuple[str, str]] = []
    pos = 0
    text = text.strip()
    while pos < len(text):
        m = _TOK.match(text, pos)
        if not m:
            break
        pos = m.end()
        if m.group(1) is not None:
            toks.append(("num", m.group(1)))
        elif m.group(2) is not None:
            toks.append(("id", m.group(2)))
        elif m.group(3).strip():
            toks.append(("op", m.group(3)))
    i = 0

    def peek():
        return toks[i] if i < len(toks) else ("end", "")

    def take():
        nonlocal i
        t = peek()
        i += 1
        return t

    def expr() -> float:
        v = term()
        while peek() in (("op", "+"), ("op", "-")):
            v = v + term() if take()[1] == "+" else v - term()
        return v

    def term() -> float:
        v = unary()
        while peek() in (("op", "*"), ("op", "/")):
            v = v * unary() if take()[1] == "*" else v / unary()
        return v

    def unary() -> float:
        if peek() == ("op", "-"):
            take()
            return -unary()
        if peek() == ("op", "+"):
            take()
            return unary()
        return power()

    def power() -> float:
        b = atom()
        if peek() == ("op", "^"):
            take()
            return b ** unary()          # right associative
        return b

    def atom() -> float:
        kind, s = take()
        if kind == "num":
            return float(s)
        if kind == "id":
            if s == "pi":
                return math.pi
            if s in _FUNCS and peek() == ("op", "("):
                take()
                v = expr()
                if take() != ("op", ")"):
                    raise ValueError("qasm: ')' expected in %r" % text)
                return _FUNCS[s](v)
            raise ValueError("qasm: unknown identifier %r in %r" % (s, text))
        if (kind, s) == ("op", "("):
            v = expr()
            if take() != ("op", ")"):
                raise ValueError("qasm: ')' expected in %r" % text)
            return v
        raise ValueError("qasm: cannot parse expression %r" % text)

    v = expr()
    if i != len(toks):
        raise ValueError("qasm: trailing input in expression %r" % text)
    return v


# ---- gate library (qelib1.inc) --------------------------------------------------------------------
def _controlled(U: np.ndarray) -> np.ndarray:
    """qubits = (control, target): local bit 0 is the control  [R2]."""
    M = np.eye(4, dtype=C128)
    M[np.ix_([1, 3], [1, 3])] = U
    return M


def _ry(t: float) -> np.ndarray:
    c, s = math.cos(0.5 * t), math.sin(0.5 * t)
    return np.array([[c, -s], [s, c]], dtype=C128)


def _swap() -> np.ndarray:
    M = np.zeros((4, 4), dtype=C128)
    for c in range(4):
        M[((c & 1) << 1) | (c >> 1), c] = 1
    return M


def _cswap() -> np.ndarray:      # qubits = (control, a, b)
    M = np.zeros((8, 8), dtype=C128)
    for c in range(8):
        r = c
        if c & 1:
            a, b = (c >> 1) & 1, (c >> 2) & 1
            r = 1 | (b << 1) | (a << 2)
        M[r, c] = 1
    return M


_Y = np.array([[0, -1j], [1j, 0]], dtype=C128)
_Z = np.diag([1, -1]).astype(C128)
_SDG = np.diag([1, -1j]).astype(C128)
_TDG = np.diag([1, complex(math.sqrt(0.5), -math.sqrt(0.5))]).astype(C128)

# name -> (number of parameters, number of qubits, builder)
GATES = {
    "U": (3, 1, lambda t, p, l: W.mat_u3(t, p, l)), "u3": (3, 1, lambda t, p, l: W.mat_u3(t, p, l)), "u": (3, 1, lambda t, p, l: W.mat_u3(t, p, l)),
    "u2": (2, 1, lambda p, l: W.mat_u3(0.5 * math.pi, p, l)), "u1": (1, 1, lambda l: W.mat_u3(0.0, 0.0, l)),
    "u0": (1, 1, lambda g: np.eye(2, dtype=C128)), "id": (0, 1, lambda: np.eye(2, dtype=C128)),
    "x": (0, 1, W.mat_x), "y": (0, 1, lambda: _Y.copy()), "z": (0, 1, lambda: _Z.copy()), "h": (0, 1, W.mat_h),
    "s": (0, 1, W.mat_s), "sdg": (0, 1, lambda: _SDG.copy()), "t": (0, 1, W.mat_t), "tdg": (0, 1, lambda: _TDG.copy()),
    "rx": (1, 1, W.mat_rx), "ry": (1, 1, _ry), "rz": (1, 1, W.mat_rz),
    "cx": (0, 2, lambda: W.mat_mcx(2)), "CX": (0, 2, lambda: W.mat_mcx(2)), "cy": (0, 2, lambda: _controlled(_Y)),
    "cz": (0, 2, lambda: W.mat_diag_minus_last(2)), "ch": (0, 2, lambda: _controlled(W.mat_h())), "swap": (0, 2, _swap),
    "ccx": (0, 3, lambda: W.mat_mcx(3)), "cswap": (0, 3, _cswap),
    "crz": (1, 2, lambda l: _controlled(W.mat_rz(l))), "cu1": (1, 2, lambda l: _controlled(W.mat_u3(0.0, 0.0, l))),
    "cu3": (3, 2, lambda t, p, l: _controlled(W.mat_u3(t, p, l))),
    "rzz": (1, 2, lambda t: np.diag([1, complex(math.cos(t), math.sin(t)), complex(math.cos(t), math.sin(t)), 1]).astype(C128)),
}


def _klass(U: np.ndarray, m: int) -> str:
    if W.is_diagonal(U):
        return "diag"
    nz = U != 0
    if np.all(nz.sum(axis=0) == 1) and np.all(nz.sum(axis=1) == 1):
        return "perm"
    return "gen%d" % m


_STMT = re.compile(r"^([A-Za-z_]\w*)\s*(?:\((.*)\))?\s*(.*)$", re.S)
_ARG = re.compile(r"^([A-Za-z_]\w*)\s*(?:\[\s*(\d+)\s*\])?$")


def _split_params(s: str) -> List[str]:
    out, depth, cur = [], 0, ""
    for ch in s:
        if ch == "," and depth == 0:
            out.append(cur)
            cur = ""
            continue
        depth += ch == "("
        depth -= ch == ")"
        cur += ch
    if cur.strip():
        out.append(cur)
    return out


def loads(text: str, name: str = "qasm") -> W.Circuit:
    """Parse OpenQASM 2.0 text into a Circuit (no truncation settings: set max_terms / min_mass on the result)."""
    text = re.sub(r"//[^\n]*", "", text)
    regs: Dict[str, Tuple[int, int]] = {}      # qreg name -> (first qubit, size)
    n = 0
    gates: List[W.Gate] = []
    seen_header = False
    for raw in text.split(";"):
        st = raw.strip()
        if not st:
            continue
        if st.startswith("OPENQASM"):
            ver = st.split()[1] if len(st.split()) > 1 else ""
            if not ver.startswith("2"):
                raise ValueError("qasm: only OPENQASM 2.x is supported, got %r" % st)
            seen_header = True
            continue
        if st.startswith("include"):
            continue
        m = _STMT.match(st)
        if not m:
            raise ValueError("qasm: cannot parse statement %r" % st)
        op, params, rest = m.group(1), m.group(2), m.group(3).strip()
        if op == "qreg":
            a = _ARG.match(rest)
            if not a or a.group(2) is None:
                raise ValueError("qasm: bad qreg %r" % st)
            if a.group(1) in regs:
                raise ValueError("qasm: register %r declared twice" % a.group(1))
            regs[a.group(1)] = (n, int(a.group(2)))
            n += int(a.group(2))
            continue
        if op in ("creg", "barrier", "measure"):
            continue
        if op in ("gate", "opaque", "if", "reset"):
            raise ValueError("qasm: %r statements are not supported (%r)" % (op, st[:40]))
        if op not in GATES:
            raise ValueError("qasm: unknown gate %r" % op)
        npar, nq, build = GATES[op]
        pv = [eval_expr(p) for p in _split_params(params)] if params is not None and params.strip() else []
        if len(pv) != npar:
            raise ValueError("qasm: gate %s takes %d parameter(s), got %d" % (op, npar, len(pv)))
        args = [x.strip() for x in rest.split(",")] if rest else []
        if len(args) != nq:
            raise ValueError("qasm: gate %s takes %d qubit(s), got %d" % (op, nq, len(args)))
        cols: List[List[int]] = []
        width = 1
        for x in args:
            a = _ARG.match(x)
            if not a or a.group(1) not in regs:
                raise ValueError("qasm: unknown qubit argument %r in %r" % (x, st))
            first, size = regs[a.group(1)]
            if a.group(2) is None:                        # whole register: broadcast
                cols.append(list(range(first, first + size)))
                if width != 1 and size != width:
                    raise ValueError("qasm: registers of different sizes in %r" % st)
                width = size
            else:
                idx = int(a.group(2))
                if idx >= size:
                    raise ValueError("qasm: index out of range in %r" % st)
                cols.append([first + idx])
        U = np.ascontiguousarray(build(*pv), dtype=C128)
        kl = _klass(U, nq)
        for r in range(width):
            qs = tuple(c[r] if len(c) > 1 else c[0] for c in cols)
            if len(set(qs)) != nq:
                raise ValueError("qasm: repeated qubit in %r" % st)
            gates.append(W.Gate(op, qs, U.copy(), kl))
    if not seen_header:
        raise ValueError("qasm: missing OPENQASM header")
    if n == 0:
        raise ValueError("qasm: no qreg")
    if n > 64:
        raise ValueError("qasm: more than 64 qubits (keys are uint64)")
    return W.Circuit(name, n, gates)


def load(path: str) -> W.Circuit:
    with open(path, "r") as f:
        return loads(f.read(), name=path)


def dumps_u3_cz(n: int, ops) -> str:
    """Write a u3 + cz circuit as OpenQASM 2.0 text in the shape of the paper's excerpt.
    ops: iterable of ("u3", q, theta, phi, lam) / ("cz", a, b)."""
    out = ["OPENQASM 2.0;", 'include "qelib1.inc";', "qreg q[%d];" % n, "creg c[%d];" % n]
    for o in ops:
        if o[0] == "u3":
            out.append("u3(%.17g,%.17g,%.17g) q[%d];" % (o[2], o[3], o[4], o[1]))
        elif o[0] == "cz":
            out.append("cz q[%d],q[%d];" % (o[1], o[2]))
        else:
            raise ValueError("dumps_u3_cz: unsupported op %r" % (o[0],))
    return "\n".join(out) + "\n"
