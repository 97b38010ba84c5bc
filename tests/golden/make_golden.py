"""Writes tests/golden/poiseuille.txt from the paper's closed form.  Calls no solver."""
import os

bx, nu, ny, dy, wall = 1.0e-3, 0.05, 32, 0.25, 2
# walls: cells j < wall and j >= ny - wall are solid; no-slip zeros sit AT the wall-adjacent solid
# cell centres y_w0 = (wall-1)*dy and y_w1 = (ny-wall)*dy, so D = y_w1 - y_w0.
y0, y1 = (wall - 1) * dy, (ny - wall) * dy
D = y1 - y0
lines = [f"# bx={bx} nu={nu} ny={ny} dy={dy} wall={wall} D={D}  U(y)=(-bx/2nu) y^2 + (bx D/2nu) y, PAPER.md:171",
         f"# bulk velocity bx D^2/(12 nu) = {bx * D * D / (12 * nu)!r}"]
for j in range(ny):
    y = j * dy - y0
    U = (-bx / (2 * nu)) * y * y + (bx * D / (2 * nu)) * y if wall <= j < ny - wall else 0.0
    lines.append(f"{j} {U!r}")
with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "poiseuille.txt"), "w") as f:
    f.write("\n".join(lines) + "\n")
