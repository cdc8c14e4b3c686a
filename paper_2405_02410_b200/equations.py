"""Equation-string front end (section III "Writing models"): host-only, no arithmetic of the method.

    m = Model(system)                       # any object with the boundary's builder calls (pss.System, the oracle's System)
    m.add_parameter("D", 1.0)
    phi = m.create_field("phi", True)
    m.add_equation("dt phi + D*q^2*phi = 0")
    m.add_noise("phi", "D")

Grammar.  A dynamic equation is ``dt <field> [+ lhs] = rhs``; an intermediate field is defined by
``lhs = rhs`` where every lhs term is linear in the field being defined.  Expressions are sums and
products of numbers, named parameters, fields, field powers ``phi^3``, parentheses and the reserved keywords
``q^2n`` (powers of -laplacian), ``iqx iqy iqz`` (derivatives, optional ``^n``) and ``1/q`` (optional ``^n``); there is an
asterisk between every pair of factors.  Division is allowed by a constant (``/2``, ``/eta``).  Since the equation is
written in Fourier space, the operators of a rhs term act on the WHOLE product of its fields.

Every term is expanded to  coef * q^(2m) * (1/q)^p * (iqx)^ax (iqy)^ay (iqz)^az * f1 * f2 ...  and handed to the boundary:
  lhs term of a dynamic equation            -> add_linear(field, op)                      (implicit, L = -lhs; reading A3)
  rhs term with one field                   -> add_term(field, op, [f])                   (explicit linear, reading A8)
  rhs term with n >= 2 fields               -> add_term(field, op, [f1..fn])
  intermediate field: lhs                   -> add_aux_lhs(aux, op)   (omitted when the lhs is the bare field)
                      rhs, one field        -> add_aux_def(aux, op, src)
                      rhs, n >= 2 fields    -> add_aux_term(aux, op, [f1..fn])
  add_noise(field, "D*q^2")                 -> set_noise(field, D, 2)
"""
import re

_TOKEN = re.compile(r"\s*(?:(\d+\.?\d*(?:[eE][-+]?\d+)?|\.\d+(?:[eE][-+]?\d+)?)|([A-Za-z_][A-Za-z_0-9]*)|(.))")
RESERVED = ("dt", "q", "iqx", "iqy", "iqz")


class EquationError(ValueError):
    pass


class _Term:
    """coef * q^(2*q2) * (1/q)^invq * prod (iq_j)^iq[j] * prod fields"""
    __slots__ = ("coef", "q2", "invq", "iq", "fields")

    def __init__(self, coef=1.0, q2=0, invq=0, iq=(0, 0, 0), fields=()):
        self.coef, self.q2, self.invq, self.iq, self.fields = float(coef), int(q2), int(invq), tuple(iq), tuple(fields)

    def mul(self, o):
        return _Term(self.coef * o.coef, self.q2 + o.q2, self.invq + o.invq,
                     tuple(a + b for a, b in zip(self.iq, o.iq)), self.fields + o.fields)

    def is_const(self):
        return self.q2 == 0 and self.invq == 0 and self.iq == (0, 0, 0) and not self.fields

    def op(self, coef=None):
        d = {"coef": self.coef if coef is None else coef}
        if self.q2:
            d["q2_pow"] = self.q2
        if self.invq:
            d["invq_pow"] = self.invq
        if any(self.iq):
            d["iq_pow"] = self.iq
        return d


def _tokens(text):
    out, pos = [], 0
    text = text.strip()
    while pos < len(text):
        m = _TOKEN.match(text, pos)
        if not m:
            break
        pos = m.end()
        if m.group(1) is not None:
            out.append(("num", m.group(1)))
        elif m.group(2) is not None:
            out.append(("id", m.group(2)))
        elif m.group(3) in "+-*/^()=":
            out.append((m.group(3), m.group(3)))
        else:
            raise EquationError("unexpected character %r in %r" % (m.group(3), text))
    return out


class _Parser:
    def __init__(self, toks, params, fields, text):
        self.t, self.i, self.params, self.fields, self.text = toks, 0, params, fields, text

    def peek(self, k=0):
        return self.t[self.i + k] if self.i + k < len(self.t) else (None, None)

    def take(self, kind=None):
        tok = self.peek()
        if tok[0] is None or (kind is not None and tok[0] != kind):
            raise EquationError("expected %s at token %d of %r" % (kind or "a token", self.i, self.text))
        self.i += 1
        return tok

    def int_power(self, what):
        """optional ^n after an operator or field; returns n (default 1)"""
        if self.peek()[0] != "^":
            return 1
        self.take("^")
        k, v = self.take("num")
        if not re.fullmatch(r"\d+", v):
            raise EquationError("%s needs a non-negative integer power in %r" % (what, self.text))
        return int(v)

    def expr(self):
        terms = []
        sign = 1.0
        if self.peek()[0] in ("+", "-"):
            sign = -1.0 if self.take()[0] == "-" else 1.0
        terms += [_Term(sign * t.coef, t.q2, t.invq, t.iq, t.fields) for t in self.product()]
        while self.peek()[0] in ("+", "-"):
            sign = -1.0 if self.take()[0] == "-" else 1.0
            terms += [_Term(sign * t.coef, t.q2, t.invq, t.iq, t.fields) for t in self.product()]
        return terms

    def product(self):
        acc = self.factor()
        while self.peek()[0] in ("*", "/"):
            if self.take()[0] == "*":
                rhs = self.factor()
                acc = [a.mul(b) for a in acc for b in rhs]
            else:
                rhs = self.factor()
                if len(rhs) != 1 or not rhs[0].is_const() or rhs[0].coef == 0.0:
                    raise EquationError("division is only allowed by a non-zero constant (and as the keyword 1/q) in %r" % self.text)
                acc = [_Term(a.coef / rhs[0].coef, a.q2, a.invq, a.iq, a.fields) for a in acc]
        return acc

    def factor(self):
        kind, val = self.peek()
        if kind == "-":
            self.take()
            return [_Term(-t.coef, t.q2, t.invq, t.iq, t.fields) for t in self.factor()]
        if kind == "+":
            self.take()
            return self.factor()
        if kind == "(":
            self.take("(")
            inner = self.expr()
            self.take(")")
            n = self.int_power("a parenthesis")
            out = [_Term()]
            for _ in range(n):
                out = [a.mul(b) for a in out for b in inner]
            return out
        if kind == "num":
            # the keyword 1/q, optionally 1/q^n
            if float(val) == 1.0 and self.peek(1)[0] == "/" and self.peek(2) == ("id", "q"):
                self.take(); self.take(); self.take()
                return [_Term(invq=self.int_power("1/q"))]
            self.take()
            return [_Term(coef=float(val))]
        if kind == "id":
            self.take()
            if val == "q":
                if self.peek()[0] != "^":
                    raise EquationError("the keyword q must be followed by ^ and an even number (PAPER.md:186) in %r" % self.text)
                n = self.int_power("q")
                if n % 2:
                    raise EquationError("q^%d: only even powers of q are operators (PAPER.md:186); use 1/q or iqx/iqy/iqz" % n)
                return [_Term(q2=n // 2)]
            if val in ("iqx", "iqy", "iqz"):
                iq = [0, 0, 0]
                iq["xyz".index(val[2])] = self.int_power(val)
                return [_Term(iq=iq)]
            if val == "dt":
                raise EquationError("dt may only open a dynamic equation (PAPER.md:184)")
            if val in self.params:
                return [_Term(coef=self.params[val])]
            if val in self.fields:
                n = self.int_power("a field")
                return [_Term(fields=(val,) * n)]
            raise EquationError("unknown name %r in %r (not a parameter, not a field)" % (val, self.text))
        raise EquationError("unexpected token %r in %r" % (val, self.text))


def _merge(terms):
    """sum terms with identical operator and field list; drop exact zeros"""
    out = {}
    order = []
    for t in terms:
        key = (t.q2, t.invq, t.iq, t.fields)
        if key not in out:
            out[key] = 0.0
            order.append(key)
        out[key] += t.coef
    return [_Term(out[k], k[0], k[1], k[2], k[3]) for k in order if out[k] != 0.0]


class Model:
    """Parser state bound to one system object (the boundary's builder calls)."""

    def __init__(self, system):
        self.s = system
        self.params = {}
        self.fields = {}      # name -> (id, dynamic)
        self.defined = set()

    # ---- PAPER.md:145-150 ----
    def add_parameter(self, name, value):
        if name in RESERVED or name in self.fields:
            raise EquationError("%r is reserved or already a field" % name)
        self.params[name] = float(value)

    def create_field(self, name, dynamic=True):
        if name in RESERVED or name in self.params or name in self.fields:
            raise EquationError("%r is reserved or already in use" % name)
        fid = self.s.add_field(name, bool(dynamic))
        self.fields[name] = (fid, bool(dynamic))
        return fid

    def ids(self):
        return {k: v[0] for k, v in self.fields.items()}

    def _parse(self, text):
        p = _Parser(_tokens(text), self.params, self.fields, text)
        e = p.expr()
        if p.peek()[0] is not None:
            raise EquationError("trailing input at token %d of %r" % (p.i, text))
        return e

    def add_equation(self, text):
        if text.count("=") != 1:
            raise EquationError("an equation has exactly one '=': %r" % text)
        left, right = (x.strip() for x in text.split("="))
        rhs = _merge(self._parse(right)) if right not in ("0", "0.0") else []
        m = re.match(r"dt\s+([A-Za-z_][A-Za-z_0-9]*)\s*(.*)$", left)
        if m:  # ---- dynamic field ----
            name, rest = m.group(1), m.group(2).strip()
            if name not in self.fields or not self.fields[name][1]:
                raise EquationError("dt %s: not a dynamic field" % name)
            if name in self.defined:
                raise EquationError("field %s already has an equation" % name)
            fid = self.fields[name][0]
            lhs = _merge(self._parse(rest)) if rest else []
            for t in lhs:
                if t.fields != (name,):
                    raise EquationError("implicit terms must be linear in %s (PAPER.md:162): %r" % (name, text))
                self.s.add_linear(fid, t.op())
            for t in rhs:
                if not t.fields:
                    raise EquationError("a rhs term without a field (a constant source) is not part of the method: %r" % text)
                self.s.add_term(fid, t.op(), [self.fields[f][0] for f in t.fields])
            self.defined.add(name)
            return fid
        # ---- intermediate field ----
        lhs = _merge(self._parse(left))
        names = {t.fields for t in lhs}
        if len(names) != 1 or len(next(iter(names))) != 1:
            raise EquationError("the lhs of an intermediate field must be linear in that one field (PAPER.md:175): %r" % text)
        name = next(iter(names))[0]
        if name not in self.fields or self.fields[name][1]:
            raise EquationError("%s is not an intermediate field" % name)
        if name in self.defined:
            raise EquationError("field %s already has an equation" % name)
        fid = self.fields[name][0]
        bare = len(lhs) == 1 and lhs[0].coef == 1.0 and lhs[0].q2 == 0 and lhs[0].invq == 0 and lhs[0].iq == (0, 0, 0)
        if not bare:
            for t in lhs:
                self.s.add_aux_lhs(fid, t.op())
        if not rhs:
            raise EquationError("an intermediate field needs a right-hand side: %r" % text)
        for t in rhs:
            if not t.fields:
                raise EquationError("a rhs term without a field is not part of the method: %r" % text)
            if name in t.fields:
                raise EquationError("%s cannot appear on its own right-hand side: %r" % (name, text))
            if len(t.fields) == 1:
                self.s.add_aux_def(fid, t.op(), self.fields[t.fields[0]][0])
            else:
                self.s.add_aux_term(fid, t.op(), [self.fields[f][0] for f in t.fields])
        self.defined.add(name)
        return fid

    # ---- PAPER.md:192-199 ----
    def add_noise(self, name, text):
        if name not in self.fields or not self.fields[name][1]:
            raise EquationError("noise needs a dynamic field, got %r" % name)
        e = _merge(self._parse(text))
        if len(e) != 1 or e[0].fields or any(e[0].iq):
            raise EquationError("a noise prefactor is a real number times a power of q^2 and 1/q (PAPER.md:194): %r" % text)
        t = e[0]
        if t.coef < 0:
            raise EquationError("negative noise strength in %r" % text)
        self.s.set_noise(self.fields[name][0], t.coef, 2 * t.q2 - t.invq)
