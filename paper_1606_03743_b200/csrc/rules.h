// The ten cubature rules of arXiv 1606.03743, Appendix A (triangles) and
// Appendix B (rectangles, L335-386), typed from the paper as ORBIT ROWS and expanded on the host
// when the library is loaded.  This file belongs to the CUDA library; the CPU oracle under
// oracle/ carries its own transcription and the two share nothing.
//
// Triangle row  {orbit, a, b, c, w}: barycentric generator (a,b,c), weight w per generated point.
//   T_ONE  : the single point (a,b,c)                               (centroid rows)
//   T_ABB  : the 3 different permutations of (a,b,b)                (L292, L309, L320)
//   T_CYC  : the 3 cyclic shifts (a,b,c),(b,c,a),(c,a,b)            (Table A3 caption, L300)
//   T_ALL  : all 6 permutations of (a,b,c)                          (L309, L320)
// Rectangle row {orbit, x, y, w}: natural coordinates in [-1,1]^2.
//   R_ONE  : (x,y)
//   R_SIGN : (+-x, +-y), all 4 sign changes                         (Tables B1-B3 captions)
//   R_AXIS : (+-x, 0) and (0, +-x)                                  (Table B3 rows 1-4)
//   R_YPM  : (0, +-y)                                               (Table B2 rows 2-3)
//   R_ROT  : (x,y), (-x,-y), (-y,x), (y,-x)                         (Tables B4/B5 captions, L364, L374)
//
// Readings of garbled cells (DESIGN.md "Readings" 1-5): Table A2's second row is blank in
// PAPER.md; it is (t+2ts, t-ts, t-ts) with weight (155+sqrt15)/1200 by the caption (L292) and the
// worked example (L127).  "S" in Tables B1-B3 is the caption's lower-case s.
#pragma once
#include <cmath>

namespace bemcub_rules {

enum TriOrbit { T_ONE, T_ABB, T_CYC, T_ALL };
enum RectOrbit { R_ONE, R_SIGN, R_AXIS, R_YPM, R_ROT };

struct TriRow { TriOrbit orbit; double a, b, c, w; };
struct RectRow { RectOrbit orbit; double x, y, w; };

static const int kNumLevels = 5;
static const int kTriN[kNumLevels] = {4, 7, 12, 19, 33};
static const int kTriDegree[kNumLevels] = {3, 5, 7, 9, 12};
static const int kRectN[kNumLevels] = {4, 7, 12, 17, 33};
static const int kRectDegree[kNumLevels] = {3, 5, 7, 9, 13};
static const int kMaxN = 33;

struct TriPoint { double la, lb, lc, w; };
struct RectPoint { double x, y, w; };

inline int tri_rows(int level, TriRow* rows) {
  const double third = 1.0 / 3.0;
  const double q15 = std::sqrt(15.0);
  switch (level) {
    case 0:  // Table A1 (L283-290)
      rows[0] = {T_ONE, third, third, third, -9.0 / 16.0};
      rows[1] = {T_ABB, 0.6, 0.2, 0.2, 25.0 / 48.0};
      return 2;
    case 1: {  // Table A2 (L292-298): t = 1/3, s = (1-sqrt15)/7, r = (1+sqrt15)/7
      const double s = (1.0 - q15) / 7.0, r = (1.0 + q15) / 7.0;
      rows[0] = {T_ONE, third, third, third, 9.0 / 40.0};
      rows[1] = {T_ABB, third * (1.0 + 2.0 * s), third * (1.0 - s), third * (1.0 - s), (155.0 + q15) / 1200.0};
      rows[2] = {T_ABB, third * (1.0 + 2.0 * r), third * (1.0 - r), third * (1.0 - r), (155.0 - q15) / 1200.0};
      return 3;
    }
    case 2:  // Table A3 (L300-307)
      rows[0] = {T_CYC, 0.06238226509439084, 0.06751786707392436, 0.8700998678316848, 0.05303405631486900};
      rows[1] = {T_CYC, 0.05522545665692000, 0.3215024938520156, 0.6232720494910644, 0.08776281742889622};
      rows[2] = {T_CYC, 0.03432430294509488, 0.6609491961867980, 0.3047265008681072, 0.05755008556995056};
      rows[3] = {T_CYC, 0.5158423343536001, 0.2777161669764050, 0.2064414986699949, 0.13498637401961758};
      return 4;
    case 3:  // Table A4 (L309-318)
      rows[0] = {T_ONE, third, third, third, 0.09713579628279610};
      rows[1] = {T_ABB, 0.02063496160252593, 0.48968251919873704, 0.48968251919873704, 0.03133470022713983};
      rows[2] = {T_ABB, 0.1258208170141290, 0.4370895914929355, 0.4370895914929355, 0.07782754100477543};
      rows[3] = {T_ABB, 0.6235929287619356, 0.18820353561903219, 0.18820353561903219, 0.07964773892720910};
      rows[4] = {T_ABB, 0.9105409732110941, 0.04472951339445297, 0.04472951339445297, 0.02557767565869810};
      rows[5] = {T_ALL, 0.03683841205473626, 0.7411985987844980, 0.22196298916076573, 0.04328353937728940};
      return 6;
    case 4:  // Table A5 (L320-331)
      rows[0] = {T_ABB, 0.4570749859701478, 0.27146250701492611, 0.27146250701492611, 0.06254121319590276};
      rows[1] = {T_ABB, 0.1197767026828138, 0.44011164865859310, 0.44011164865859310, 0.04991833492806094};
      rows[2] = {T_ABB, 0.0235924981089169, 0.48820375094554155, 0.48820375094554155, 0.02426683808145203};
      rows[3] = {T_ABB, 0.7814843446812914, 0.10925782765935432, 0.10925782765935432, 0.02848605206887754};
      rows[4] = {T_ABB, 0.9507072731273288, 0.02464636343633558, 0.02464636343633558, 0.00793164250997364};
      rows[5] = {T_ALL, 0.1162960196779266, 0.2554542286385173, 0.62824975168355610, 0.04322736365941421};
      rows[6] = {T_ALL, 0.02303415635526714, 0.2916556797383410, 0.68531016390639186, 0.02178358503860756};
      rows[7] = {T_ALL, 0.02138249025617059, 0.1272797172335894, 0.85133779251024000, 0.01508367757651144};
      return 8;
  }
  return 0;
}

inline int rect_rows(int level, RectRow* rows) {
  switch (level) {
    case 0: {  // Table B1 (L335-342): s = 1/sqrt3
      const double s = 1.0 / std::sqrt(3.0);
      rows[0] = {R_SIGN, s, s, 0.25};
      return 1;
    }
    case 1: {  // Table B2 (L344-351): t = sqrt(14/15), r = sqrt(3/5), s = sqrt(1/3)
      rows[0] = {R_ONE, 0.0, 0.0, 2.0 / 7.0};
      rows[1] = {R_YPM, 0.0, std::sqrt(14.0 / 15.0), 5.0 / 63.0};
      rows[2] = {R_SIGN, std::sqrt(3.0 / 5.0), std::sqrt(1.0 / 3.0), 5.0 / 36.0};
      return 3;
    }
    case 2: {  // Table B3 (L353-362)
      const double q = std::sqrt(583.0);
      rows[0] = {R_AXIS, std::sqrt(6.0 / 7.0), 0.0, 49.0 / 810.0};
      const double s = std::sqrt((114.0 - 3.0 * q) / 287.0), t = std::sqrt((114.0 + 3.0 * q) / 287.0);
      rows[1] = {R_SIGN, s, s, (178981.0 + 2769.0 * q) / 1888920.0};
      rows[2] = {R_SIGN, t, t, (178981.0 - 2769.0 * q) / 1888920.0};
      return 3;
    }
    case 3:  // Table B4 (L364-372)
      rows[0] = {R_ONE, 0.0, 0.0, 0.131687242798353921};
      rows[1] = {R_ROT, 0.968849966361977720, 0.630680119731668854, 0.022219844542549678};
      rows[2] = {R_ROT, 0.750277099978900533, 0.927961645959569667, 0.028024900532399120};
      rows[3] = {R_ROT, 0.523735820214429336, 0.453339821135647190, 0.099570609815517519};
      rows[4] = {R_ROT, 0.076208328192617173, 0.852615729333662307, 0.067262834409945196};
      return 5;
    case 4:  // Table B5 (L374-386)
      rows[0] = {R_ONE, 0.0, 0.0, 0.075095528857806335};
      rows[1] = {R_ROT, 0.778809711554419422, 0.983486682439872263, 0.007497959716124783};
      rows[2] = {R_ROT, 0.957297699786307365, 0.859556005641638928, 0.009543605329270918};
      rows[3] = {R_ROT, 0.138183459862465353, 0.958925170287534857, 0.015106230954437494};
      rows[4] = {R_ROT, 0.941327225872925236, 0.390736216129461000, 0.019373184633276336};
      rows[5] = {R_ROT, 0.475808625218275905, 0.850076673699748575, 0.029711166825148901};
      rows[6] = {R_ROT, 0.755805356572081436, 0.647821637187010732, 0.032440887592500675};
      rows[7] = {R_ROT, 0.696250078491749413, 0.070741508996444936, 0.053335395364297350};
      rows[8] = {R_ROT, 0.342716556040406789, 0.409304561694038843, 0.064217687370491966};
      return 9;
  }
  return 0;
}

// Expands one level into its full point list; returns the number of points.
inline int tri_points(int level, TriPoint* out) {
  TriRow rows[8];
  const int nr = tri_rows(level, rows);
  int n = 0;
  for (int i = 0; i < nr; ++i) {
    const TriRow& r = rows[i];
    switch (r.orbit) {
      case T_ONE: out[n++] = {r.a, r.b, r.c, r.w}; break;
      case T_ABB:
        out[n++] = {r.a, r.b, r.b, r.w};
        out[n++] = {r.b, r.a, r.b, r.w};
        out[n++] = {r.b, r.b, r.a, r.w};
        break;
      case T_CYC:
        out[n++] = {r.a, r.b, r.c, r.w};
        out[n++] = {r.b, r.c, r.a, r.w};
        out[n++] = {r.c, r.a, r.b, r.w};
        break;
      case T_ALL: {
        const double v[3] = {r.a, r.b, r.c};
        static const int perm[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};
        for (int p = 0; p < 6; ++p) out[n++] = {v[perm[p][0]], v[perm[p][1]], v[perm[p][2]], r.w};
        break;
      }
    }
  }
  return n;
}

inline int rect_points(int level, RectPoint* out) {
  RectRow rows[9];
  const int nr = rect_rows(level, rows);
  int n = 0;
  for (int i = 0; i < nr; ++i) {
    const RectRow& r = rows[i];
    switch (r.orbit) {
      case R_ONE: out[n++] = {r.x, r.y, r.w}; break;
      case R_SIGN:
        for (int sx = 1; sx >= -1; sx -= 2)
          for (int sy = 1; sy >= -1; sy -= 2) out[n++] = {sx * r.x, sy * r.y, r.w};
        break;
      case R_AXIS:
        out[n++] = {r.x, 0.0, r.w};
        out[n++] = {-r.x, 0.0, r.w};
        out[n++] = {0.0, r.x, r.w};
        out[n++] = {0.0, -r.x, r.w};
        break;
      case R_YPM:
        out[n++] = {0.0, r.y, r.w};
        out[n++] = {0.0, -r.y, r.w};
        break;
      case R_ROT:
        out[n++] = {r.x, r.y, r.w};
        out[n++] = {-r.x, -r.y, r.w};
        out[n++] = {-r.y, r.x, r.w};
        out[n++] = {r.y, -r.x, r.w};
        break;
    }
  }
  return n;
}

}  // namespace bemcub_rules
