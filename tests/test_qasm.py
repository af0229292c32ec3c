"""OpenQASM 2.0 reader (paper_2607_07816_b200/qasm.py).  CPU only.
Pins: expression values typed out, gate matrices against the qelib1 definitions written here independently (products of
U(theta, phi, lambda) and CX), register broadcast, and whole circuits through the dense simulator of oracle/."""
import cmath
import math

import numpy as np
import pytest

from paper_2607_07816_b200 import qasm, workloads as W
from oracle import dense

HDR = 'OPENQASM 2.0;\ninclude "qelib1.inc";\n'


def u3_ref(t, p, l):
    """qelib1: U(theta, phi, lambda) = [[cos(t/2), -e^{il} sin(t/2)], [e^{ip} sin(t/2), e^{i(p+l)} cos(t/2)]]."""
    return np.array([[math.cos(t / 2), -cmath.exp(1j * l) * math.sin(t / 2)],
                     [cmath.exp(1j * p) * math.sin(t / 2), cmath.exp(1j * (p + l)) * math.cos(t / 2)]])


@pytest.mark.parametrize("text,want", [
    ("pi/2", math.pi / 2), ("-pi/4", -math.pi / 4), ("3*pi/8", 3 * math.pi / 8), ("2^3", 8.0), ("2^-1", 0.5), ("-2^2", -4.0),
    ("sin(pi/6)", 0.5), ("cos(0)+ln(exp(2))", 3.0), ("sqrt(16)/(1+1)", 2.0), ("1.5e-3", 0.0015), (".25*4", 1.0), ("(1-(2-3))", 2.0),
    ("0.30000000000000004", 0.30000000000000004),
])
def test_expressions(text, want):
    assert qasm.eval_expr(text) == pytest.approx(want, rel=1e-15, abs=1e-15)


@pytest.mark.parametrize("bad", ["pi pi", "2*", "foo(1)", "(1", "1)"])
def test_expression_errors(bad):
    with pytest.raises(ValueError):
        qasm.eval_expr(bad)


def test_single_qubit_gates_against_qelib1_definitions():
    t, p, l = 0.7, -1.1, 2.3
    c = qasm.loads(HDR + "qreg q[1];\nu3(%r,%r,%r) q[0]; u2(%r,%r) q[0]; u1(%r) q[0]; U(%r,%r,%r) q[0];" % (t, p, l, p, l, l, t, p, l))
    ref = [u3_ref(t, p, l), u3_ref(math.pi / 2, p, l), u3_ref(0, 0, l), u3_ref(t, p, l)]
    for g, r in zip(c.gates, ref):
        assert np.allclose(g.U, r, atol=1e-15)
    # named gates as qelib1 writes them in terms of u1 / u2 / u3 (up to the global phase of rx / ry / rz)
    named = {"x": u3_ref(math.pi, 0, math.pi), "y": u3_ref(math.pi, math.pi / 2, math.pi / 2), "z": u3_ref(0, 0, math.pi),
             "h": u3_ref(math.pi / 2, 0, math.pi), "s": u3_ref(0, 0, math.pi / 2), "sdg": u3_ref(0, 0, -math.pi / 2),
             "t": u3_ref(0, 0, math.pi / 4), "tdg": u3_ref(0, 0, -math.pi / 4), "id": np.eye(2)}
    for nm, r in named.items():
        g = qasm.loads(HDR + "qreg q[1]; %s q[0];" % nm).gates[0]
        assert np.allclose(g.U, r, atol=1e-15), nm
    a = 0.9
    for nm, r in {"rx": u3_ref(a, -math.pi / 2, math.pi / 2), "ry": u3_ref(a, 0, 0), "rz": u3_ref(0, 0, a)}.items():
        g = qasm.loads(HDR + "qreg q[1]; %s(%r) q[0];" % (nm, a)).gates[0]
        k = np.argmax(np.abs(r.ravel()))
        ph = g.U.ravel()[k] / r.ravel()[k]
        assert abs(abs(ph) - 1) < 1e-15 and np.allclose(g.U, ph * r, atol=1e-15), nm


def _circuit_matrix(c):
    """Columns = images of the basis states under the dense simulator of oracle/ (itself pinned to Kronecker products)."""
    d = 1 << c.n
    M = np.zeros((d, d), dtype=np.complex128)
    for col in range(d):
        psi = np.zeros(d, dtype=np.complex128)
        psi[col] = 1
        for g in c.gates:
            psi = dense.apply_gate(psi, c.n, g.qubits, g.U)
        M[:, col] = psi
    return M


def test_two_and_three_qubit_gates_against_their_qelib1_decompositions():
    """qelib1 defines cz, cy, ch, swap, ccx, crz, cu1, cu3, cswap, rzz as products of CX and one-qubit gates: the built-in
    matrix and the decomposition (typed from the standard library's definitions) must be the same operator up to a phase."""
    decomp = {
        "cz a,b": "h b; cx a,b; h b;",
        "cy a,b": "sdg b; cx a,b; s b;",
        "swap a,b": "cx a,b; cx b,a; cx a,b;",
        "ccx a,b,c": "h c; cx b,c; tdg c; cx a,c; t c; cx b,c; tdg c; cx a,c; t b; t c; h c; cx a,b; t a; tdg b; cx a,b;",
        "cswap a,b,c": "cx c,b; ccx a,b,c; cx c,b;",
        "crz(0.8) a,b": "u1(0.4) b; cx a,b; u1(-0.4) b; cx a,b;",
        "cu1(0.8) a,b": "u1(0.4) a; cx a,b; u1(-0.4) b; cx a,b; u1(0.4) b;",
        # (with the u1 on the control that makes it the controlled U(theta, phi, lambda) exactly, not up to a phase on the control)
        "cu3(0.5,0.3,-0.9) a,b": "u1((0.3+-0.9)/2) a; u1((-0.9-0.3)/2) b; cx a,b; u3(-0.5/2,0,-(0.3+-0.9)/2) b; cx a,b; u3(0.5/2,0.3,0) b;",
        "rzz(0.6) a,b": "cx a,b; u1(0.6) b; cx a,b;",
        "ch a,b": "h b; sdg b; cx a,b; h b; t b; cx a,b; t b; h b; s b; x b; s a;",
    }
    regs = "qreg a[1]; qreg b[1]; qreg c[1];"
    for gate, seq in decomp.items():
        A = _circuit_matrix(qasm.loads(HDR + regs + gate + ";"))
        B = _circuit_matrix(qasm.loads(HDR + regs + seq))
        k = np.argmax(np.abs(B.ravel()))
        ph = A.ravel()[k] / B.ravel()[k]
        assert abs(abs(ph) - 1) < 1e-12 and np.allclose(A, ph * B, atol=1e-12), gate


def test_registers_broadcast_and_ignored_statements():
    c = qasm.loads(HDR + "// a comment\nqreg a[2];\nqreg b[2];\ncreg m[4];\nh a;\ncx a,b;\ncx a[1],b;\nbarrier a,b;\nmeasure a -> m;\n")
    assert c.n == 4
    assert [(g.name, g.qubits) for g in c.gates] == [("h", (0,)), ("h", (1,)), ("cx", (0, 2)), ("cx", (1, 3)), ("cx", (1, 2)), ("cx", (1, 3))]
    assert [g.klass for g in c.gates] == ["gen1", "gen1", "perm", "perm", "perm", "perm"]
    assert qasm.loads(HDR + "qreg q[2]; cz q[0],q[1]; rz(0.1) q[1];").gates[0].klass == "diag"


@pytest.mark.parametrize("bad", [
    "qreg q[2]; h q[0];",                                # no header
    HDR + "h q[0];",                                     # no register
    HDR + "qreg q[2]; foo q[0];", HDR + "qreg q[2]; cx q[0],q[0];", HDR + "qreg q[2]; h q[2];", HDR + "qreg q[2]; rx q[0];",
    HDR + "qreg q[2]; cx q[0];", HDR + "qreg q[1]; gate g a { h a; } g q[0];", HDR + "qreg q[1]; creg c[1]; if(c==1) x q[0];",
    "OPENQASM 3.0; qubit[2] q;", HDR + "qreg q[65]; h q[0];", HDR + "qreg a[2]; qreg b[3]; cx a,b;",
])
def test_errors(bad):
    with pytest.raises(ValueError):
        qasm.loads(bad)


def test_ghz_through_the_dense_simulator():
    n = 5
    c = qasm.loads(HDR + "qreg q[%d];\nh q[0];\n" % n + "".join("cx q[%d],q[%d];\n" % (i, i + 1) for i in range(n - 1)))
    psi = dense.run(c.n, c.gates)
    want = np.zeros(1 << n, dtype=np.complex128)
    want[0] = want[-1] = math.sqrt(0.5)
    assert np.allclose(psi, want, atol=1e-15)


def test_ring_circuit_round_trip_in_the_shape_of_the_papers_excerpt():
    """A u3 + cz ring (own seeded angles, the shape of PAPER.md:150-171) written as QASM text and read back: the same
    gate list as the records built directly, bit for bit (%.17g round-trips a double)."""
    rng = np.random.default_rng(11)
    n = 6
    ops, direct = [], []
    for layer in range(2):
        for a in range(layer % 2, n - 1 + layer % 2, 2):
            b = (a + 1) % n
            ta, tb = float(rng.uniform(0, math.pi)), float(rng.uniform(0, math.pi))
            ops += [("u3", a, ta, 0.0, -0.5 * math.pi), ("u3", b, tb, 0.0, 0.5 * math.pi), ("cz", a, b)]
            direct += [((a,), W.mat_u3(ta, 0.0, -0.5 * math.pi)), ((b,), W.mat_u3(tb, 0.0, 0.5 * math.pi)), ((a, b), W.mat_diag_minus_last(2))]
    text = qasm.dumps_u3_cz(n, ops)
    assert text.startswith("OPENQASM 2.0;") and "u3(" in text and "cz q[" in text
    c = qasm.loads(text)
    assert c.n == n and len(c.gates) == len(direct)
    for g, (qs, U) in zip(c.gates, direct):
        assert g.qubits == qs and np.array_equal(g.U, U)
