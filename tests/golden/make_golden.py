"""Re-derives the golden fixtures from first principles with `math` only (no oracle, no CUDA path).

Run: python tests/golden/make_golden.py   (prints the values stored in the .txt files next to it)
"""
import math

PHI_M1_5 = 0.0668072012688581     # standard normal CDF at -1.5 (normal tables)
PHI_3 = 0.9986501019683699        # standard normal CDF at 3.0


def main():
    # P4: z=[1,2], a=[3], W1=[[1,0,-1],[2,1,0]], b1=[.5,-1]  => u = [1-3+.5, 2+2-1] = [-1.5, 3]
    u = [-1.5, 3.0]
    g = [u[0] * PHI_M1_5, u[1] * PHI_3]
    # W2=[[1,1],[0,2]], b2=[.25,-.5]:  v = z + W2 g + b2
    v = [1 + g[0] + g[1] + 0.25, 2 + 2 * g[1] - 0.5]
    m = (v[0] + v[1]) / 2
    var = ((v[0] - m) ** 2 + (v[1] - m) ** 2) / 2
    ln = [(x - m) / math.sqrt(var + 1e-5) for x in v]
    print("p4 gelu", g, "v", v, "ln", ln)
    # P5
    x = [1.0, 2.0, 3.0, 4.0]
    for eps in (0.0, 1e-5):
        print("p5", eps, [(xi - 2.5) / math.sqrt(1.25 + eps) for xi in x])
    # P6
    sig = lambda t: 1 / (1 + math.exp(-t))
    z = [1.0, -2.0]
    gate = [sig(2.0), sig(-3.0)]
    r = [sig(-2.0), sig(1.0)]
    rz = [r[0] * z[0], r[1] * z[1]]
    h = [math.tanh(rz[0] + rz[1] + 0.5), math.tanh(rz[0] - rz[1] + 1.0)]
    zn = [(1 - gate[i]) * z[i] + gate[i] * h[i] for i in range(2)]
    print("p6 g", gate, "r", r, "h", h, "z'", zn)
    # P14 (TransH step, PAPER.md:164 / DESIGN.md S24): z=[3,4], a=[2], W_w=[[1],[0]], W_d=[[.5],[-1]], eps=1e-12
    eps = 1e-12
    uw = [2.0, 0.0]
    nw = math.sqrt(uw[0] ** 2 + uw[1] ** 2 + eps)
    w = [uw[0] / nw, uw[1] / nw]
    dot = w[0] * 3.0 + w[1] * 4.0
    x = [3.0 - dot * w[0] + 1.0, 4.0 - dot * w[1] - 2.0]          # z_perp + W_d a  (= [1, 2] up to eps)
    # W1=[[1,0,-1.25],[2,1,-.5]], b1=[0,0] => u = [x0 - 2.5, 2 x0 + x1 - 1] (= [-1.5, 3] up to eps)
    u = [x[0] - 2.5, 2 * x[0] + x[1] - 1.0]
    phi = lambda t: 0.5 * (1.0 + math.erf(t / math.sqrt(2.0)))
    g = [u[0] * phi(u[0]), u[1] * phi(u[1])]
    v = [x[0] + g[0] + g[1] + 0.25, x[1] + 2 * g[1] - 0.5]        # W2=[[1,1],[0,2]], b2=[.25,-.5]
    nv = math.sqrt(v[0] ** 2 + v[1] ** 2 + eps)
    print("p14 x", x, "v", v, "z'", [v[0] / nv, v[1] / nv])


if __name__ == "__main__":
    main()
