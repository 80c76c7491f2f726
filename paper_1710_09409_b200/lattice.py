"""Expression-template front end in the spirit of the paper's Listings 1-3: `z.assign(x*y + v)`.
Operators on Lattice objects only BUILD a tree (no arithmetic happens in Python); `assign` flattens the tree to the
postfix program of su3_expr, with every distinct field as one operand, and the library evaluates it in one pass.
Argument marshalling only."""
from . import Field, su3_expr


class Expr:
    def __init__(self, op, a, b):
        self.op, self.a, self.b = op, a, b

    def __add__(self, o):
        return Expr("+", self, _node(o))

    def __sub__(self, o):
        return Expr("-", self, _node(o))

    def __mul__(self, o):
        return Expr("*", self, _node(o))


class Lattice(Expr):
    """a field (matrix or real scalar kind) that can appear in expressions and be assigned to"""

    def __init__(self, field: Field):
        self.field = field

    def assign(self, expr, stream=None):
        prog, operands = postfix(_node(expr))
        su3_expr(self.field, prog, [l.field for l in operands], stream=stream)
        return self


def _node(x):
    if isinstance(x, Expr):
        return x
    raise TypeError("expressions are built from Lattice objects (got %r)" % type(x).__name__)


def postfix(expr):
    """(program string, list of distinct Lattice operands in order of first use)"""
    operands, out = [], []

    def walk(e):
        if isinstance(e, Lattice):
            for k, l in enumerate(operands):
                if l is e:
                    break
            else:
                operands.append(e)
                k = len(operands) - 1
            if k > 7:
                raise ValueError("more than 8 distinct fields in one expression")
            out.append(str(k))
        else:
            walk(e.a)
            walk(e.b)
            out.append(e.op)
    walk(expr)
    return "".join(out), operands
